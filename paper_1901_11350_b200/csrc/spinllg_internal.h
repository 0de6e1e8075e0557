// spinllg_internal.h -- private definitions of the B200 LLG library (not part of the C-ABI).
//
// Layout in HBM: spins are kept structure-of-arrays and sublattice-major,
//     n[b*sub + ((ic+LC)*PB + (ib+LB)) * 3*PA + comp*PA + (ia+LA)],   comp in {x,y,z}      (see DevicePlan)
// so that a warp reads 32 consecutive doubles of one component of one lattice row (256 B, two full lines), the three
// components of a row are adjacent, and ghost cells make every neighbour a constant offset from the own site.
// The boundary order (AoS, basis fastest; include/spinllg.h) is converted by pack/unpack kernels.
#pragma once

#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/spinllg.h"

#define SPIN_MAX_BASIS 8
#define SPIN_MAX_PAIR_ENTRIES 160
#define SPIN_MAX_QUAD_ENTRIES 32
#define SPIN_MAX_ANI_ENTRIES 16      // anisotropy axes over all basis atoms
#define SPIN_COOP_MAX_SPINS 4096      // largest lattice that takes the cooperative all-steps kernel by default

namespace spin {

// CODATA 2018 (reading R5)
constexpr double MU_B = 0.057883818060;    // meV / T
constexpr double K_B = 0.08617333262;      // meV / K
constexpr double GAMMA = 0.176085963023;   // rad / (ps T)
constexpr double C_DD = 0.0536815112;      // meV, mu0 mu_B^2 / (4 pi Angstrom^3)

enum TermMask { T_ZEE = 1, T_ANI = 2, T_EXC = 4, T_DMI = 8, T_QUAD = 16, T_DDI = 32, T_ALL = 63 };

// One gather entry of a basis atom's pair table: the spin at cell c collects J n_j + n_j x D from the partner
// on sublattice bj at cell c + (da,db,dc).  Backward entries carry -D and -t ("unique pairs").
struct PairEntry {
    int da, db, dc;      // partner cell translation, reduced to (-N_d, N_d) in periodic directions
    int bj;              // partner sublattice
    int lin;             // linear index offset valid when no coordinate wraps (interior bricks)
    int pad_;
    double J, Dx, Dy, Dz;
};

// One role of one quadruplet (Eq. 2): F += K (n_Q . n_R) n_P, the three other members given relative to this spin.
struct QuadEntry {
    int d[3][3];         // translations of P, Q, R relative to this spin
    int b[3];            // their sublattices
    int lin[3];
    int pad_;
    double K;
};

struct DevicePlan {
    int Na, Nb, Nc;
    int perA, perB, perC;
    int nb;
    int Ncell;
    // ---- Layout of every per-spin array (n, n^p, A, dipolar force), in doubles:
    //   index(b, ia, ib, ic, comp) = b*sub + ((ic+LC)*PB + (ib+LB)) * 3*PA + comp*PA + (ia+LA)
    // i.e. sublattice-major, then rows of the padded lattice, each row holding its x, y and z components as three
    // consecutive runs of PA doubles (component offset PA*8 bytes: an immediate in the load instruction).
    // rA/rB/rC ghost cells on each side hold the periodic images (gA/gB/gC = 1) or zeros (open edges).
    // LA and PA are multiples of 16 doubles so that every run starts on a 128-byte line.
    int LA, LB, LC;
    int PA, PB, PC;
    int sub;                                 // 3*PA*PB*PC
    int rA, rB, rC;                          // ghost width: the reach (max |translation| per direction over all table entries) times ghost_mult
    int ghost_mult;                          // 1, or 2 when the one-pass plane-marching kernel is in use (its rim predictor reads n two reaches out)
    int gA, gB, gC;                          // periodic images to maintain in that direction
    int pair_begin[SPIN_MAX_BASIS + 1];
    int quad_begin[SPIN_MAX_BASIS + 1];
    double zee[SPIN_MAX_BASIS][3];           // mu_b mu_B B            (meV)
    int ani_begin[SPIN_MAX_BASIS + 1];       // anisotropy entries of basis atom b: [ani_begin[b], ani_begin[b+1])  (Eq. 1 sums over axes)
    double K2[SPIN_MAX_ANI_ENTRIES];         // 2 K of the entry       (meV)
    double Kax[SPIN_MAX_ANI_ENTRIES][3];     // its unit axis
    double pre[SPIN_MAX_BASIS];              // -gamma / ((1+alpha^2) mu_b mu_B)   (rad / (ps meV))
    double sigma[SPIN_MAX_BASIS];            // thermal amplitude sqrt(2 alpha kB T mu / (gamma dt)) (meV)
    double inv_mu[SPIN_MAX_BASIS];           // 1 / (mu_b mu_B)        (T / meV)
    double alpha, dt, dt2;
    int stt_on;
    int has_ddi;
    int cell_off;                            // slab decomposition: global cell index of local cell 0 (the thermal field is keyed by the GLOBAL spin)
    double stt_c[3];                         // j^ = sum_d stt_c[d] a_d   (1/Angstrom)
    double stt_s, stt_x;                     // -u (alpha-beta)/(1+alpha^2),  u (1+alpha beta)/(1+alpha^2)
    uint32_t seed_lo, seed_hi;
    int thermal_on;
    int damping_only;                        // 1: the precession term of Eq. 10 is dropped (:168)
    const unsigned char *pin;                // N flags in boundary order (b + nb*cell) or null: pinned spins are never updated
    const double *mu_ratio;                  // N ratios mu_i / mu_b(i) in boundary order or null: per-site moments ("atoms of different types")
    PairEntry pairs[SPIN_MAX_PAIR_ENTRIES];
    QuadEntry quads[SPIN_MAX_QUAD_ENTRIES];
};

struct HostPair { int bi, bj, t[3]; double J, D[3]; };
struct HostQuad { int b[4]; int t[9]; double K; };

}  // namespace spin

struct DdiState;   // spin_ddi.cu
struct JitState;   // spin_jit.cu

struct spin_system {
    // ---- geometry
    double brav[9];
    int nb;
    std::vector<double> basis;     // 3*nb fractional
    int nc[3], per[3];
    double alat;
    int64_t ncell, N;
    // ---- Hamiltonian (host description)
    std::vector<double> mu;        // nb
    double Bmag, Bdir[3];
    std::vector<int> ani_b;        // anisotropy entries: basis atom,
    std::vector<double> K, Kax;    // strength, unit axis (3 per entry)
    std::vector<spin::HostPair> pairs_explicit, pairs_exch_shells, pairs_dmi_shells;
    std::vector<spin::HostQuad> quads;
    int ddi_on, ddi_img[3];
    // ---- LLG
    double dt_ps, alpha, T, u, jdir[3], beta;
    uint64_t seed, step;
    int solver;                    // SPIN_SOLVER_*
    int damping_only;              // drop the precession term (minimisation with the LLG solvers, :168)
    // ---- device
    cudaStream_t stream, own_stream;
    double *d_n[2];                // ping-pong spin buffers (nb*sub doubles each)
    int cur;
    double *d_np;                  // predictor
    double *d_A;                   // rotation field of the predictor stage (store_A option)
    double *d_fddi[2];             // dipolar force of n and of n^p (nb*sub doubles each), only with DDI
    double *d_aos;                 // staging buffer, boundary order (3N)
    double *d_partials;            // reduction scratch
    double *d_result;              // reduction result (16 doubles)
    unsigned long long *d_step;    // device copy of the step counter (read by the kernels)
    unsigned char *d_pin;          // pinned-spin flags (boundary order), null if none
    std::vector<double> mu_site;   // per-site moments in mu_B (boundary order), empty if none
    double *d_mu_ratio;            // mu_i / mu_b(i) on the device (rebuilt with the plan: the basis moments may change), null if none
    // ---- slab decomposition along c over several GPUs: this system holds planes [slab_off, slab_off + nc[2]) of a
    // lattice of slab_gnc planes; its ghost layers along c are filled by the halo exchange, not by its own periodic images
    int slab_on, slab_off, slab_gnc, slab_gper;
    // ---- batched images: n_img independent configurations of the same lattice and Hamiltonian; every per-spin array holds them
    // one after the other (stride nb * plan.sub doubles); the sweeps take the image from blockIdx.z
    int n_img, img_sel;            // number of images; image that spins_set/get, effective_field, energy, ... address
    double *d_img_sigma;           // per-image factor on the thermal amplitude, sqrt(T_image / T), or null (all 1)
    std::vector<double> img_T;     // the absolute per-image temperatures it was made from (empty: none set)
    unsigned int *d_bar;           // arrival counter of the cooperative kernel's grid barrier
    unsigned long long *d_flags;   // step flags of a slab (spin_slab_flags): [0] written by the lower, [1] by the upper neighbour
    double *d_vp;                  // velocity-projection state: ratio r, started flag, |F|^2
    bool vp_active;                // d_A holds the force of the previous VP iteration
    int vp_cur;                    // which of {d_A, d_fddi[1]} holds it
    spin::DevicePlan plan;
    bool plan_dirty;
    DdiState *ddi;
    JitState *jit;                 // run-time specialised sweeps (null: table-driven kernels)
    bool has_device;               // false only in the planner-only mode used by the CPU tests
    std::string jit_note;          // why the specialised sweeps are not in use, if they are not
    // ---- execution options / bookkeeping
    int opt_graph, opt_store_A, opt_jit, opt_ddi_slab, opt_ddi_mirror, opt_pdl, opt_cache_noise, opt_coop, opt_march;
    cudaGraphExec_t graph_exec[2];   // one captured graph per ping-pong parity
    int graph_steps;
    int64_t graph_launches;    // kernel launches of one replay of the captured graph (counted while capturing)
    int64_t n_launch, n_fft;
    int profile_on;
    double prof_ms[4];             // predictor, corrector, dipolar evaluation (whole), dipolar contraction kernel alone
    int64_t prof_n[4];
    cudaEvent_t ev2, ev3;          // around the dipolar contraction kernel (inside the evaluation that ev0/ev1 bracket)
    cudaEvent_t ev0, ev1;
};

namespace spin {
// shared error plumbing (spin_api.cu)
int fail(int code, const char *fmt, ...);
#define SPIN_CUDA(call)                                                                             \
    do {                                                                                            \
        cudaError_t e__ = (call);                                                                   \
        if (e__ != cudaSuccess)                                                                     \
            return spin::fail(SPIN_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), \
                              __FILE__, __LINE__);                                                  \
    } while (0)

// spin_ddi.cu
int ddi_prepare(spin_system *s);                                   // (re)build tensor spectra and FFT plans
int ddi_field(spin_system *s, const double *d_n, double *d_f);     // d_f (SoA, meV) = dipolar force of d_n
void ddi_release(spin_system *s);
bool ddi_graph_ok(const spin_system *s);                              // the evaluation is kernels of this library only (no cuFFT call)
const char *ddi_path_name(const spin_system *s);                      // "off", "3d", "slab", "slab+mirror"

// spin_jit.cu
std::string jit_source(const spin_system *s);
int jit_compile(const std::string &source, std::string &cubin, std::string &log);
std::string jit_compiler_info();      // version and path of the NVRTC in use
int jit_prepare(spin_system *s);
void jit_release(spin_system *s);
bool jit_ready(const spin_system *s);
const char *jit_log(const spin_system *s);
// one stage of the RK4 solver (jit_rk4_stage)
int jit_launch_rk4_stage(spin_system *s, const double *base, const double *y, double *ynext, double *acc, double *noise, const double *fddi,
                         int stage, unsigned step_add);
// the whole Depondt step in one pass (jit_depondt_march, spin_jit_march.cuh): 3-D lattices of one basis atom without dipolar coupling
bool march_eligible(const spin_system *s);      // spin_api.cu: decided from the system alone (the planner doubles the ghost layers for it)
bool jit_march_ready(const spin_system *s);
int jit_launch_march(spin_system *s, int cur, double *nout, unsigned step_add, int part = 0, double *peer_lo = nullptr, double *peer_hi = nullptr,
                     int peer_lo_nc = 0);
// all steps of an llg_iterate call in one cooperative launch (jit_steps_coop)
bool jit_coop_ready(const spin_system *s);
bool jit_cluster_ready(const spin_system *s);
int jit_launch_steps_coop(spin_system *s, unsigned nsteps);
int jit_launch_predictor(spin_system *s, dim3 grid, dim3 block, const double *n, const double *fddi, double *np, double *Aout,
                         unsigned step_add, unsigned brick0 = 0, unsigned nbricks = 0);
int jit_launch_corrector(spin_system *s, dim3 grid, dim3 block, const double *n, const double *np, const double *fddi_n,
                         const double *fddi_np, const double *Ain, double *nout, unsigned step_add, unsigned brick0 = 0, unsigned nbricks = 0);
void jit_brick_shape(const spin_system *s, int b[3]);
}  // namespace spin
