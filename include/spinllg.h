/*
 * spinllg.h -- C-ABI boundary of the B200-native LLG hot path.
 *
 * One data-parallel path of "Spirit: Multifunctional Framework for Atomistic Spin Simulations"
 * (arXiv 1901.11350; line numbers below are /root/reference/PAPER.md):
 *
 *     n  ->  F(n) = -dH/dn  (extended Heisenberg Hamiltonian, Eq. 1 :61-67 and Eq. 2 :75)
 *        ->  Depondt predictor/corrector update of every spin (Eq. 10 :147-153, App. B B5-B7 :369-380)
 *
 * Every step of the path runs in hand-written CUDA kernels for sm_100a (cuFFT performs only the
 * Fourier transforms of the dipolar convolution).  There is no CPU fallback: every call that needs the
 * device returns SPIN_ERR_CUDA when no CUDA device is usable.
 *
 * Conventions
 *   units       energy meV, field Tesla, moments mu_B, time fs at the API (ps inside), length Angstrom
 *   constants   CODATA 2018: mu_B = 0.057883818060 meV/T, k_B = 0.08617333262 meV/K,
 *               gamma = 0.176085963023 rad/(ps T), mu0 mu_B^2/(4 pi A^3) = 0.0536815112 meV
 *   spin index  i = b + n_basis*(ia + Na*(ib + Nb*ic)), b the basis atom (fastest), (ia,ib,ic) the cell
 *   arrays      "host" pointers are ordinary host memory owned by the caller; "device" pointers are
 *               CUDA device memory owned by the caller.  All spin / field arrays at the boundary are
 *               AoS: x0 y0 z0 x1 y1 z1 ... (3N doubles).  The internal layout is private.
 *   ownership   the library owns all memory behind spin_system; setters copy, getters copy
 *   errors      every function returns 0 (SPIN_OK) or a negative code; nothing throws across the ABI;
 *               spin_last_error() gives a message for the last failure on the calling thread
 *   ordering    setters may be called in any order; the device plan is (re)built lazily by the next
 *               call that computes
 *   streams     all device work of a system is enqueued on one CUDA stream (default: a private
 *               non-blocking stream); spin_set_stream() rebinds it, e.g. to torch's current stream
 */
#ifndef SPINLLG_H
#define SPINLLG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spin_system spin_system;

enum {
    SPIN_OK = 0,
    SPIN_ERR_ARG = -1,        /* bad argument (null pointer, out-of-range index, self pair, ...) */
    SPIN_ERR_STATE = -2,      /* call not valid in this state                                    */
    SPIN_ERR_MEMORY = -3,     /* host or device allocation failed                                */
    SPIN_ERR_CUDA = -4,       /* CUDA / cuFFT error, or no device                                */
    SPIN_ERR_LIMIT = -5       /* interaction table larger than the kernels support               */
};

/* ---- geometry (PAPER.md:79 "Bravais vectors and basis cells with any given number of atoms"; :307 boundary
 * conditions).  bravais: rows a, b, c in units of lattice_constant_A.  basis_frac: 3*n_basis fractional
 * coordinates.  n_cells >= 1 each.  periodic: 0 = open, 1 = periodic per direction.  A 2-D lattice is
 * n_cells[2] = 1 with periodic[2] = 0.  Initial state: all spins +z, mu_s = 1, no interactions.
 * 1 <= n_basis <= 8, N = n_basis*prod(n_cells) < 2^31.                                                      */
int spin_geometry_create(const double bravais[9], int n_basis, const double *basis_frac /*host*/,
                         const int n_cells[3], const int periodic[3], double lattice_constant_A,
                         spin_system **out);
void spin_system_destroy(spin_system *sys);
int64_t spin_system_nspins(const spin_system *sys);

/* Bind the CUDA stream (a cudaStream_t passed as void*; NULL = back to the system's private stream).
 * The legacy default stream cannot be captured into CUDA graphs and is not accepted. */
int spin_set_stream(spin_system *sys, void *cuda_stream);

/* ---- Hamiltonian, Eq. 1 (:61-67) and Eq. 2 (:75) ------------------------------------------------------- */
/* magnetic moments mu_i per basis atom, in mu_B, > 0 (":59 m_i = mu_i n_i") */
int hamiltonian_set_mu_s(spin_system *sys, const double *mu_s /*host, n_basis*/);
/* ":79 defects, such as vacancies and atoms of different types": one moment per SITE (host, N values in mu_B in boundary order, > 0),
 * replacing the basis atom's wherever mu_i enters -- the Zeeman term and the dipolar sum of Eq. 1, the 1/mu_i of Eq. 10, the thermal
 * amplitude of Eq. 11 and the conversion of effective_field to Tesla.  NULL goes back to the basis atoms' moments.  The array is copied.
 * Costs one extra 8-byte read per spin and sweep.                                                                                  */
int hamiltonian_set_site_mu_s(spin_system *sys, const double *mu_site /*host, N, or NULL*/);
/* Zeeman term -sum_i mu_i B.n_i: field magnitude in Tesla and direction (normalised internally) */
int hamiltonian_set_field(spin_system *sys, double B_tesla, const double dir[3]);
/* uniaxial anisotropy -sum_i sum_j K_j (K^_j.n_i)^2 (Eq. 1 :61, ":69 axes ... of the basis cell"): n entries (basis_idx, K_meV, axis);
 * a basis atom may be listed several times (several axes j, e.g. the biaxial Hamiltonian of Eq. 13 :187), atoms not listed
 * have none; a later call replaces the earlier one; at most 16 entries in total                                              */
int hamiltonian_set_anisotropy(spin_system *sys, int n, const int *basis_idx, const double *K_meV,
                               const double *axis /*host, 3n*/);
/* unique pairs <ij> (":69 unique pairs", ":71 no limitation on number or distance"): pair p couples basis atom
 * i_basis[p] in cell c with j_basis[p] in cell c + translation[p], with -J n_i.n_j - D.(n_i x n_j).
 * Each bond is listed ONCE (either direction); D_ji = -D_ij is implied.  D_meV may be NULL (no DMI).
 * Errors: index out of range, a pair of a site with itself (same basis atom, zero translation).
 * Replaces any earlier explicit pair list (shell helpers below are kept separately and add up).             */
int hamiltonian_set_pairs(spin_system *sys, int n_pairs, const int *i_basis, const int *j_basis,
                          const int *translation /*host, 3*n_pairs*/, const double *J_meV,
                          const double *D_meV /*host, 3*n_pairs or NULL*/);
/* helper: exchange by neighbour shell; shell s (s = 0 nearest) gets J_meV[s] on all of its bonds.  The host
 * neighbour finder only scans directions with n_cells > 1.                                                  */
int hamiltonian_set_exchange_shells(spin_system *sys, int n_shells, const double *J_meV);
/* helper: DMI by neighbour shell with a direction convention (the paper leaves D_ij to the user):
 * chirality +1/-1: D_ij = +/- D r^_ij (bulk, Bloch);  +2/-2: D_ij = +/- D (z^ x r^_ij) (interfacial, Neel)    */
int hamiltonian_set_dmi_shells(spin_system *sys, int n_shells, const double *D_meV, int chirality);
/* quadruplets, Eq. 2: -K (n_i.n_j)(n_k.n_l); basis_ijkl: 4 basis atoms per quadruplet; translation_jkl: cell
 * translations of j, k, l relative to i (9 ints per quadruplet).  Sites may repeat (4-spin-2-site, 3-site).  */
int hamiltonian_set_quadruplets(spin_system *sys, int n, const int *basis_ijkl /*host, 4n*/,
                                const int *translation_jkl /*host, 9n*/, const double *K_meV);
/* dipole-dipole coupling through the zero-padded FFT convolution (:81-87).  n_periodic_images[d]: images
 * t_d in [-n, n] summed in periodic direction d (ignored in open directions).                               */
int hamiltonian_set_ddi(spin_system *sys, int enabled, const int n_periodic_images[3]);

/* ---- state ---------------------------------------------------------------------------------------------- */
/* spins are normalised on input; a zero vector is an error except on a pinned site (a vacancy, see spins_set_pinned) */
int spins_set(spin_system *sys, const double *n_xyz /*host, 3N AoS*/);
int spins_get(spin_system *sys, double *n_xyz /*host, 3N AoS*/);
int spins_set_device(spin_system *sys, const double *n_xyz /*device, 3N AoS*/);
int spins_get_device(spin_system *sys, double *n_xyz /*device, 3N AoS*/);

/* ---- batched images (":197 chain of images", temperature sweeps of Fig. 13): n_images independent configurations of the same lattice
 * and Hamiltonian advance in the same launches (the sweeps take the image from the third grid dimension).  New images start as
 * copies of image 0.  Image m draws its thermal noise from the Philox counter words block + 2 m, at its own temperature if
 * llg_set_image_temperatures gives one (host array of n_images Kelvin values; needs T > 0 in llg_configure; NULL: all at T).
 * spin_select_image chooses the image that spins_set/get[_device], effective_field, energy, observables and topological_charge
 * address (default 0).  Two-stage solvers only; minimise_vp and the RK4 solver work on a single image (SPIN_ERR_STATE).     */
int spin_set_images(spin_system *sys, int n_images);
int spin_select_image(spin_system *sys, int image);
int llg_set_image_temperatures(spin_system *sys, const double *T_kelvin /*host, n_images, or NULL*/);

/* Geodesic nudged elastic band on the batched images (III.D Eqs. 14-17 :193-216, App. F :475-489): the images are a chain, image 0
 * and image n_images-1 its fixed ends.  Per interior image: tangent by the definitions of Ref. 55 (energy-weighted forward/backward
 * differences), projected on the tangent space spin by spin (F1) and normalised in 3N dimensions; spring force kappa (l_{nu,nu+1} -
 * l_{nu-1,nu}) tau with geodesic distances l (Eq. 15); gradient force -grad E + (grad E . tau) tau (Eq. 16); for the climbing image
 * (index, or -1 for none) no spring and -grad E + 2 (grad E . tau) tau (Eq. 17); the total projected per spin (F2).
 * gneb_forces returns F (host, n_images x 3N AoS, zero for the ends), the energies and l[nu] = l_{nu,nu+1}; any may be NULL.
 * gneb_iterate relaxes the chain: x <- x + step F, renormalised, n_iterations times (step in 1/meV).  Blocking calls.        */
int gneb_forces(spin_system *sys, double kappa, int climbing_image, double *F_xyz, double *E_meV, double *l_geodesic);
int gneb_iterate(spin_system *sys, int64_t n_iterations, double step, double kappa, int climbing_image);

/* Pinning and vacancies (:79 "pinning of individual spins or a set of spins", "defects, such as vacancies").  mask: N flags in
 * boundary index order, non-zero = pinned; NULL removes all pins.  A pinned spin is never updated by llg_iterate but acts on its
 * neighbours as usual.  A vacancy is a pinned site holding the zero vector: spins_set accepts a zero vector on pinned sites only;
 * such a site contributes nothing to any field or energy.  Pinned sites are excluded from the max-torque observable.
 * Call before spins_set if the configuration contains vacancies.                                                              */
int spins_set_pinned(spin_system *sys, const unsigned char *mask /*host, N*/);

/* ---- dynamics: Eq. 10 with the thermal field of Eq. 11 (:157-160), Depondt solver (App. B) --------------
 * dt in fs; alpha Gilbert damping; T in Kelvin (0 = no noise); seed of the counter-based Philox4x32-10
 * generator keyed by (seed; step, spin, block); u in Angstrom/ps along the unit vector j_dir; beta the
 * non-adiabatic parameter.  Resets the step counter to 0.                                                   */
int llg_configure(spin_system *sys, double dt_fs, double alpha, double T_kelvin, uint64_t seed,
                  double u_A_per_ps, const double j_dir[3], double beta);
/* Solver of the LLG equation written as dn/dt = n x A (B1, :349).  All are two-stage predictor/corrector schemes over the same
 * two field sweeps and share the thermal field of the step between the stages:
 *   SPIN_SOLVER_DEPONDT  App. B, B5-B7 (:369-380): rotations R(A), renormalised                       (default)
 *   SPIN_SOLVER_HEUN     App. B, B3-B4 (:355-367): n + dt/2 (n x A + n^p x A^p), renormalised every step
 *   SPIN_SOLVER_SIB      App. C, C5-C11 (:384-436): semi-implicit midpoint; field of the corrector at {(n_j + n_j^p)/2};
 *                        preserves |n_i| by construction (no renormalisation)
 *   SPIN_SOLVER_RK4      classical 4th-order Runge-Kutta (:168, named only): four field sweeps per step, renormalised every step
 * Heun, SIB and RK4 run in the run-time specialised kernels only (SPIN_ERR_STATE from llg_iterate if those are unavailable). */
enum { SPIN_SOLVER_DEPONDT = 0, SPIN_SOLVER_HEUN = 1, SPIN_SOLVER_SIB = 2, SPIN_SOLVER_RK4 = 3 };
int llg_set_solver(spin_system *sys, int solver);
/* ":168 These methods can also be used for energy minimization by considering only the damping part of the LLG equation": with
 * enabled != 0 the precession term -gamma/((1+alpha^2) mu) F of the rotation field is dropped and only the damping term remains. */
int llg_set_damping_only(spin_system *sys, int enabled);
/* advance n_steps steps of the selected solver (Depondt unless llg_set_solver chose another); asynchronous on the system's stream.  The step counter persists, so
 * llg_iterate(a); llg_iterate(b) reproduces llg_iterate(a+b) exactly.                                       */
int llg_iterate(spin_system *sys, int64_t n_steps);
int llg_get_step(const spin_system *sys, uint64_t *step);
int llg_set_step(spin_system *sys, uint64_t step);
/* Velocity-projection minimiser, App. D (:438-463), Eqs. D1-D5 with the force F_i = -dH/dn_i in meV (D4): per iteration the force
 * of the current configuration, v <- v + dt/(2m)(F_old + F) (D2), the projection of v on F over all 3N components (D3), x <- x +
 * dt v + dt^2/(2m) F (D1), renormalisation (D5).  dt and mass are the pseudo-time step and mass of that fictitious dynamics (dt^2/m
 * in 1/meV).  Velocity and previous force persist between calls; spins_set*, llg_iterate, any setter or minimise_vp_reset clear them.
 * Pinned spins do not move and carry no force.  Asynchronous on the system's stream.                                            */
int minimise_vp(spin_system *sys, int64_t n_iterations, double dt, double mass);
int minimise_vp_reset(spin_system *sys);
/* wait for all work enqueued on the system's stream */
int spin_synchronize(spin_system *sys);

/* ---- observables ------------------------------------------------------------------------------------------
 * effective_field: deterministic B_eff,i = -(1/(mu_i mu_B)) dH/dn_i in Tesla (:155), no noise, no current   */
int effective_field(spin_system *sys, double *B_xyz /*host, 3N AoS*/);
int effective_field_device(spin_system *sys, double *B_xyz /*device, 3N AoS*/);
/* total energy and its terms (Zeeman, anisotropy, exchange, DMI, quadruplet, dipolar), meV; either may be NULL */
int energy(spin_system *sys, double *E_total_meV, double E_terms_meV[6]);
/* M = (1/N) sum_i n_i (:131) and max_i |F_i - (F_i.n_i) n_i| in meV                                        */
int observables(spin_system *sys, double M[3], double *max_torque_meV);

/* topological charge of App. A (:317-343), Eqs. A1-A2: Q = (1/4 pi) sum of the signed spherical-triangle areas over the two
 * elementary triangles (r, r+a, r+a+b), (r, r+a+b, r+b) of every cell, counter-clockwise about +z, summed over the a-b planes.
 * One basis atom (SPIN_ERR_ARG otherwise).  Periodic directions wrap; triangles leaving an open edge are skipped (:343).  */
int topological_charge(spin_system *sys, double *Q);

/* The same quantity for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): topological_charge allocates and frees a buffer of per-block partial sums on every call; this variant keeps them in a
 * fixed array in device memory (128 KB per GPU that loads the library, held until exit) and calls no cudaMalloc, cudaFree or
 * allocating library routine.  It launches two kernels on the system's stream and returns without synchronising.
 *   d_Q   DEVICE pointer to one double, owned by the caller; written by the second kernel (valid after spin_synchronize or after
 *         later work on the system's stream)
 * Limits and errors: at most 4,194,304 cells (SPIN_ERR_LIMIT beyond that: use topological_charge); the system's plan must be built
 * already, because building it allocates (SPIN_ERR_STATE: call spins_set, effective_field, topological_charge or llg_iterate once
 * after the last change of the lattice, Hamiltonian or options); one basis atom (SPIN_ERR_ARG); the device that was current when
 * the system was created must be current (SPIN_ERR_STATE).
 * ALL calls on one GPU share the one array: calls that overlap on the GPU (two systems on different streams) race on it; calls
 * on the same stream, or ordered by events, are safe.  Nothing in the array has to start at zero: each call overwrites the
 * entries it reads.                                                                                                        */
int topological_charge_noalloc(spin_system *sys, double *d_Q);

/* ---- slab decomposition along c over several GPUs (SURVEY 8(e); the paper has no counterpart: MPI only as a scripting remark, :143) ----
 * One process per GPU holds `n_cells[2]` consecutive planes of a lattice of `global_cells_c` planes, starting at plane `c_offset`.  Its
 * ghost layers along c (as wide as the Hamiltonian reaches along c) are then NOT its own periodic images but its neighbours' boundary
 * planes, delivered by a halo exchange before every sweep (twice per step: n, then n^p); translations along c are folded with the global
 * extent and boundary condition, and the thermal field is keyed by the GLOBAL spin index, so N slabs reproduce the single-GPU trajectory
 * bit for bit.  The library provides the pieces below; paper_1901_11350_b200/slab.py orders them and owns the transport
 * (torch.distributed / NCCL, or device copies between slabs of one process).  Not with the dipolar term (its transform needs all-to-all
 * transposes), batched images, RK4, or a current with a component along c.                                                          */
int spin_set_slab(spin_system *sys, int enabled, int c_offset, int global_cells_c, int global_periodic_c);
/* doubles held by one side of the halo: reach along c x padded plane x sublattices (contiguous, sublattice-major); reach_c (may be
 * NULL) receives the reach = number of planes per side                                                                              */
int spin_halo_doubles(spin_system *sys, int64_t *doubles_per_side, int *reach_c);
/* array: 0 the current configuration n, 1 the predictor n^p, 2 the next configuration (corrector output, before llg_slab_advance);
 * side: 0 towards lower c, 1 towards higher c.  get copies the outermost OWN planes of that side to dst (DEVICE pointer); put copies src
 * (DEVICE pointer) into the GHOST planes of that side.  Enqueued on cuda_stream (NULL: the system's stream), never synchronised.     */
int spin_halo_get(spin_system *sys, int array, int side, double *dst_device, void *cuda_stream);
int spin_halo_put(spin_system *sys, int array, int side, const double *src_device, void *cuda_stream);
/* one sweep of the current step over part of the slab: stage 0 predictor, 1 corrector; part 0 all bricks, 1 the brick layers a neighbour
 * needs (within reach of either face), 2 the layers in between (launched while the halos of part 1 travel)                          */
int llg_slab_sweep(spin_system *sys, int stage, int part);
/* after the corrector sweeps: the next configuration becomes current, the step counter (noise stream) advances by one             */
int llg_slab_advance(spin_system *sys);
/* The whole step of a slab in ONE pass (the plane-marching kernel; available when spin_kernel_info reports "jit+march": one basis
 * atom, Depondt or Heun, no pinned spins or per-site moments, slab of at least 32 x 8 x 8 cells): the kernel recomputes the predictor of the
 * neighbours' boundary planes itself, so a step needs ONE halo exchange of depth 2 x reach (of the new configuration, array 2, before
 * llg_slab_advance) instead of two of depth reach.  spin_halo_doubles reports the depth in use.  part 0: the whole slab; 1: the first and
 * last chunk of planes, which hold everything the neighbours need; 2: the chunks in between (launched after the halo copies of part 1
 * have been started, they run while the halos travel).  SPIN_ERR_STATE if the kernel does not apply to this system (use llg_slab_sweep). */
int llg_slab_step(spin_system *sys, int part);
/* The one-pass step with the halo exchange FUSED into the kernel: it writes the boundary planes of the next configuration straight into
 * the neighbours' ghost layers, so no halo copy and no message follow a step.
 *   peer_lo_next / peer_hi_next   DEVICE pointers to the NEXT-configuration arrays of the lower / upper neighbour (from its
 *                                 spin_slab_arrays), writable from this GPU: peer access over NVLink, an opened CUDA IPC handle, or
 *                                 another system on this device; NULL where there is no neighbour (open end).  Not owned.
 *   peer_lo_cells_c               planes of the lower neighbour's slab (slabs may differ by one plane)
 * The driver keeps ORDER only: the call must be enqueued after both neighbours' previous step has completed (they wrote this slab's ghost
 * layers, and they read the arrays this step writes into).  Same conditions and errors as llg_slab_step.                    */
int llg_slab_step_fused(spin_system *sys, double *peer_lo_next, int peer_lo_cells_c, double *peer_hi_next);
/* device pointers of the current and the next configuration array of a slab (they swap at every llg_slab_advance); valid until the
 * plan is rebuilt.  Owned by the system.                                                                                   */
int spin_slab_arrays(spin_system *sys, double **current, double **next);
/* The fused exchange between PROCESSES (one per GPU).  Memory: spin_ipc_export gives the 64-byte CUDA IPC handle of the allocation that
 * holds a device pointer (a slab's arrays, its flags) and the pointer's offset in it; the neighbour's process maps it with spin_ipc_open
 * (peer access is enabled on the way) and unmaps it with spin_ipc_close.  Order: events of another process cannot carry a step number, so
 * each slab owns two flags in device memory (spin_slab_flags: [0] written by its lower, [1] by its upper neighbour, zero at first);
 * spin_flag_signal enqueues, on the system's stream, a store of `value` into a flag (release, system scope: after everything enqueued
 * before it), spin_flag_wait enqueues a wait until a flag holds at least `value` (a one-thread kernel that polls; after 30 s it traps
 * instead of hanging; every kernel that is to run while a wait polls must have run once before -- its first launch may load code,
 * which waits for the device).  A step k + 1 follows wait(own flags >= k) and is followed by signal(neighbours' flags = k + 1).  The waits depend
 * on another GPU's progress: ranks that use them must not share a GPU.                                                      */
int spin_ipc_export(const void *device_ptr, unsigned char handle[64], int64_t *offset);
int spin_ipc_open(const unsigned char handle[64], int64_t offset, void **device_ptr);
int spin_ipc_close(void *device_ptr, int64_t offset);
int spin_slab_flags(spin_system *sys, unsigned long long **flags);
int spin_flag_signal(spin_system *sys, unsigned long long *flag, unsigned long long value);
int spin_flag_wait(spin_system *sys, const unsigned long long *flag, unsigned long long value);

/* ---- execution options ------------------------------------------------------------------------------------------------
 * spin_set_option(name, value) changes how the path is executed, never what it computes (every combination is bit-identical; tested).
 * The defaults are the measured choices; the options exist for A/B measurements and for the tests.
 *   use_jit     (1)  the sweeps are specialised per system at run time with NVRTC -- lattice extents, gather tables and prefactors become
 *                    compile-time constants; 0: the table-driven kernels (also taken, with the reason kept, when NVRTC is unavailable)
 *   use_graph   (1)  16 steps are captured once into a CUDA graph and replayed (no host work per step)
 *   use_coop    (1)  lattices of up to 4096 spins without dipolar coupling run ALL steps of an llg_iterate call in one launch: as one
 *                    thread-block cluster with its hardware barrier between the sweeps (up to 16 bricks), else as a cooperative launch
 *                    with a grid barrier; 2 forces the path for any size, 3 forces the grid barrier, 0 switches it off
 *   use_pdl     (-1) programmatic dependent launch of the brick sweeps (griddepcontrol.wait inside the kernel): -1 automatic, 0 off,
 *                    1 dependents released at entry, 2 at the end of each block; any value but 0 also launches the kernels of the
 *                    fused dipolar path that way (their prologue overlaps the previous kernel's tail)
 *   store_A     (0)  1: the predictor stores the rotation field A(n) and the corrector reads it instead of recomputing it
 *   cache_noise (1)  the predictor keeps the thermal field of the step (24 B/spin) for the corrector instead of generating it twice
 *   use_march   (1)  lattices of one basis atom, 3-D (>= 32 x 8 x 8 cells) or flat (one plane), from 65536 spins on, advanced by Depondt or Heun
 *                    without dipolar coupling take the one-pass kernel: the whole step in one launch, n^p never written to memory; 0: brick sweeps;
 *                    2: also for smaller lattices (tests)
 *   ddi_slab    (1)  thin films (up to 8 planes; 4 with several basis atoms) take the dipolar slab path: hand-written transforms along a and, for one
 *                    basis atom and power-of-two columns, one fused kernel for the transforms along b and c and the contraction;
 *                    3: cuFFT's transform along b and a separate contraction kernel; 2: cuFFT's transforms along a and b; 0: the general
 *                    3-D transform
 *   ddi_mirror  (1)  the slab contraction reads PZ/2 + 1 tensor planes when the spectrum is mirror symmetric along c; 0: all PZ planes    */
int spin_set_option(spin_system *sys, const char *name, int value);

/* ==== MEASUREMENT SUPPORT ===========================================================================================
 * Nothing below is needed to use the library.  bench.py and the tests read these to say which kernels ran, how often and how long.  */
/* number of kernel launches (own kernels) and cuFFT executions issued by this system so far */
int spin_launch_counts(const spin_system *sys, int64_t *own_kernels, int64_t *cufft_execs);
/* per-kernel device timing: when enabled, CUDA events bracket the launches of the step kernels (plain launches, no graph, no
 * all-steps-in-one-launch path); get returns the accumulated milliseconds and launch counts for kind = 0 predictor, 1 corrector,
 * 2 one dipolar evaluation (all its stages), 3 the dipolar contraction kernel alone (slab path).                                 */
int spin_profile_enable(spin_system *sys, int enabled);
int spin_profile_get(spin_system *sys, int kind, double *total_ms, int64_t *launches);
/* measured fp64 FMA throughput of this device in TFLOP/s (register-only kernel, best of 5): the ALU ceiling next to the HBM one */
int spin_measure_fp64_tflops(spin_system *sys, double *tflops);
/* which sweep kernels are in use: "jit+cluster", "jit+coop", "jit (brick sweeps)" or "generic: <why>"                              */
int spin_kernel_info(spin_system *sys, char *buf, int len);
/* Which dipolar path the plan chose: "off", "3d" (general zero-padded 3-D transform) or "slab" (thin film of 1-8 planes, or 1-4 planes with several basis atoms:
 * transforms in the a-b plane, hand-written transform along c fused with the tensor contraction), followed by "+mirror" when the
 * contraction reads PZ/2 + 1 of the PZ tensor planes (spectrum found mirror symmetric along c) and by "+own-a" when the transform along a
 * is the hand-written one (rows of power-of-two length) instead of cuFFT's.                                                        */
int spin_ddi_info(spin_system *sys, char *buf, int len);
/* The run-time compiler of the specialised sweeps, e.g. "12.9 (/usr/local/cuda/lib64/libnvrtc.so.12)".  NVRTC is bound at run time by
 * path -- $SPINLLG_NVRTC, then the toolkit the library was built with, then the loader's libnvrtc.so.12 -- so that a different NVRTC
 * already loaded into the process (torch ships 12.8) does not change the generated kernels.  No device needed.  */
int spin_jit_compiler_info(char *buf, int len);
/* the generated translation unit of the specialised sweeps (buf may be NULL); compile != 0 also compiles it for sm_100a
 * (needs no device) and returns the cubin size.  Host-side planner check; works in planner-only mode
 * (environment SPINLLG_PLANNER_ONLY=1 lets spin_geometry_create succeed without a device; every computing call then
 * still fails with SPIN_ERR_CUDA).                                                                                    */
int spin_jit_source(spin_system *sys, char *buf, int len, int compile, int64_t *cubin_bytes);

const char *spin_last_error(void);
const char *spin_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPINLLG_H */
