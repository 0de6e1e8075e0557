// spin_jit_kernels.cuh -- the two Depondt sweeps specialised per spin system (compiled at run time by NVRTC for sm_100a).
//
// The host planner (spin_jit.cu) prints the system as compile-time constants into `namespace spec` and then includes this
// file.  Everything that the table-driven kernels (spin_kernels.cuh) look up at run time is a constant here:
//   * lattice extents, ghost-cell layout          -> div/mod by constants; every partner is `own address + immediate`
//   * the gather table of every basis atom        -> fully unrolled, J and D folded into fma operands, zero D components dropped
//   * LLG prefactors, time step, noise amplitude
// Ghost cells (spinllg_internal.h "Layout") hold the periodic images or, at open edges, zeros, so the gather needs neither
// wrap arithmetic nor edge tests; the writers of n^p and n(t+dt) also write the periodic images.
// One thread per spin, bricks of BX x BY x BZ spins of one sublattice per block; no atomics, no shared memory.
// Device-only: no host headers (NVRTC).  Formulas and paper citations: see spin_kernels.cuh / spin_device_math.cuh.
//
// namespace spec must define (all constexpr):
//   int NA, NB, NC, NBASIS, BX, BY, BZ;  int LA, LB, LC, PA, PB, PC, SUB, RA, RB, RC;  bool GA, GB, GC, PER_A, PER_B, PER_C;
//   bool STORE_A, HAS_DDI, THERMAL_ON, STT_ON, HAS_PIN, HAS_SITE_MU;
//   int PAIR_BEGIN[NBASIS+1], P_DA[], P_DB[], P_DC[], P_BJ[];  double P_J[], P_DX[], P_DY[], P_DZ[];
//   int QUAD_BEGIN[NBASIS+1], Q_D[][9], Q_B[][3];  double Q_K[];
//   int ANI_BEGIN[NBASIS+1];  double ZEE[NBASIS][3], K2[n_ani], KAX[n_ani][3], PRE[NBASIS], SIGMA[NBASIS];
//   double ALPHA, DT, DT2, STT_C[3], STT_S, STT_X;
#pragma once

#define SPIN_BOUNDS(t) __launch_bounds__(t)
#include "spin_device_math.cuh"

namespace spinjit {

typedef unsigned int u32;
typedef unsigned long long u64;

template <int V> struct Int { static constexpr int value = V; };

template <int I, int END, class F>
__device__ __forceinline__ void static_for(F &&f) {
    if constexpr (I < END) {
        f(Int<I>{});
        static_for<I + 1, END>(f);
    }
}

struct Coord { int ia, ib, ic; };

constexpr int ROW = 3 * spec::PA;                 // doubles between consecutive lattice rows
constexpr int PLANE = 3 * spec::PA * spec::PB;    // doubles between consecutive lattice planes

// linear offset of the partner (sublattice BJ at translation DA, DB, DC) from a site of sublattice B
template <int B, int BJ, int DA, int DB, int DC>
__host__ __device__ constexpr int lin() {
    return (BJ - B) * spec::SUB + DC * PLANE + DB * ROW + DA;
}

// q points at the x component of the own site; O is a compile-time offset in doubles
// CG = true: coherent L1-cached loads (ld.global.ca) for the cooperative kernel, in which other blocks rewrite the arrays between
// grid barriers -- the acquire fence of the barrier invalidates L1, after which weak loads must observe the released stores; the
// non-coherent read-only path (ld.global.nc, __ldg) is only legal for data nobody writes during the kernel
template <int O, bool CG = false>
__device__ __forceinline__ void load3(const double *__restrict__ q, double (&v)[3]) {
    if constexpr (CG) {
        v[0] = __ldca(q + O); v[1] = __ldca(q + O + spec::PA); v[2] = __ldca(q + O + 2 * spec::PA);
    } else {
        v[0] = __ldg(q + O); v[1] = __ldg(q + O + spec::PA); v[2] = __ldg(q + O + 2 * spec::PA);
    }
}
__device__ __forceinline__ void store3(double *__restrict__ q, const double (&v)[3]) {
    q[0] = v[0]; q[spec::PA] = v[1]; q[2 * spec::PA] = v[2];
}
// the periodic images of a spin in the ghost layers (at most one image per direction)
__device__ __forceinline__ void store_images(double *__restrict__ q, const Coord &c, const double (&v)[3]) {
    if constexpr (spec::GA || spec::GB || spec::GC) {
        // one unsigned compare per direction decides whether the site has any image at all (interior sites: nearly all)
        bool edge = false;
        if constexpr (spec::GA) { if constexpr (spec::NA > 2 * spec::RA) edge |= (unsigned)(c.ia - spec::RA) >= (unsigned)(spec::NA - 2 * spec::RA); else edge = true; }
        if constexpr (spec::GB) { if constexpr (spec::NB > 2 * spec::RB) edge |= (unsigned)(c.ib - spec::RB) >= (unsigned)(spec::NB - 2 * spec::RB); else edge = true; }
        if constexpr (spec::GC) { if constexpr (spec::NC > 2 * spec::RC) edge |= (unsigned)(c.ic - spec::RC) >= (unsigned)(spec::NC - 2 * spec::RC); else edge = true; }
        if (edge) {
            int sa = 0, sb = 0, sc = 0;
            if constexpr (spec::GA) { if (c.ia < spec::RA) sa = spec::NA; else if (c.ia >= spec::NA - spec::RA) sa = -spec::NA; }
            if constexpr (spec::GB) { if (c.ib < spec::RB) sb = spec::NB * ROW; else if (c.ib >= spec::NB - spec::RB) sb = -spec::NB * ROW; }
            if constexpr (spec::GC) { if (c.ic < spec::RC) sc = spec::NC * PLANE; else if (c.ic >= spec::NC - spec::RC) sc = -spec::NC * PLANE; }
#pragma unroll
            for (int m = 1; m < 8; ++m) {
                if (((m & 1) && !sa) || ((m & 2) && !sb) || ((m & 4) && !sc)) continue;
                store3(q + (((m & 1) ? sa : 0) + ((m & 2) ? sb : 0) + ((m & 4) ? sc : 0)), v);
            }
        }
    }
}
__device__ __forceinline__ void store_spin(double *__restrict__ q, const Coord &c, const double (&v)[3]) {
    store3(q, v);
    store_images(q, c, v);
}

// Site accessors: where the partner (sublattice BJ at translation DA, DB, DC) of a site of sublattice B is read from.
// GlobalAcc: the ghost-cell arrays in global memory (own address + immediate).
template <int NCONF, bool CG = false>
struct GlobalAcc {
    const double *cfg[NCONF];      // x component of the own site in configuration k
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int k, double (&v)[3]) const { load3<lin<B, BJ, DA, DB, DC>(), CG>(cfg[k], v); }
};

// SIB corrector (C11): the field is evaluated at the midpoint configuration {(n_j + n_j^p)/2}
template <bool CG = false>
struct MidAcc {
    const double *a, *b;           // own site in n and in n^p
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int, double (&v)[3]) const {
        double u[3], w[3];
        load3<lin<B, BJ, DA, DB, DC>(), CG>(a, u);
        load3<lin<B, BJ, DA, DB, DC>(), CG>(b, w);
        v[0] = 0.5 * (u[0] + w[0]); v[1] = 0.5 * (u[1] + w[1]); v[2] = 0.5 * (u[2] + w[2]);
    }
};

// F += (Zeeman + anisotropy + pairs + quadruplets) of basis atom B for NCONF configurations sharing the lattice
// zr: mu_i / mu_b of the site when per-site moments are set (spec::HAS_SITE_MU), the Zeeman force scales with it
template <int B, int NCONF, class Acc>
__device__ __forceinline__ void force(const Acc &cfg, const double (&own)[NCONF][3], double (&F)[NCONF][3], const double zr = 1.0) {
#pragma unroll
    for (int k = 0; k < NCONF; ++k) {
        // spec:: holds the values as constexpr (zero terms vanish at compile time); specc:: holds the same values in constant
        // memory, from where an fp64 instruction reads them as an operand (a 64-bit immediate would cost two extra moves)
        if constexpr (spec::HAS_SITE_MU) {
            if constexpr (spec::ZEE[B][0] != 0.0) F[k][0] = fma(zr, specc::ZEE[B][0], F[k][0]);
            if constexpr (spec::ZEE[B][1] != 0.0) F[k][1] = fma(zr, specc::ZEE[B][1], F[k][1]);
            if constexpr (spec::ZEE[B][2] != 0.0) F[k][2] = fma(zr, specc::ZEE[B][2], F[k][2]);
        } else {
            if constexpr (spec::ZEE[B][0] != 0.0) F[k][0] += specc::ZEE[B][0];
            if constexpr (spec::ZEE[B][1] != 0.0) F[k][1] += specc::ZEE[B][1];
            if constexpr (spec::ZEE[B][2] != 0.0) F[k][2] += specc::ZEE[B][2];
        }
        static_for<spec::ANI_BEGIN[B], spec::ANI_BEGIN[B + 1]>([&](auto ae) {      // every anisotropy axis of this atom (Eq. 1 sums over axes)
            constexpr int A = decltype(ae)::value;
            if constexpr (spec::K2[A] != 0.0) {
                constexpr bool hx = spec::KAX[A][0] != 0.0, hy = spec::KAX[A][1] != 0.0, hz = spec::KAX[A][2] != 0.0;
                double p = 0.0;
                if constexpr (hx) p = fma(specc::KAX[A][0], own[k][0], p);
                if constexpr (hy) p = fma(specc::KAX[A][1], own[k][1], p);
                if constexpr (hz) p = fma(specc::KAX[A][2], own[k][2], p);
                p *= specc::K2[A];
                if constexpr (hx) F[k][0] = fma(p, specc::KAX[A][0], F[k][0]);
                if constexpr (hy) F[k][1] = fma(p, specc::KAX[A][1], F[k][1]);
                if constexpr (hz) F[k][2] = fma(p, specc::KAX[A][2], F[k][2]);
            }
        });
    }
    static_for<spec::PAIR_BEGIN[B], spec::PAIR_BEGIN[B + 1]>([&](auto e) {
        constexpr int E = decltype(e)::value;
        constexpr double J = spec::P_J[E], Dx = spec::P_DX[E], Dy = spec::P_DY[E], Dz = spec::P_DZ[E];
#pragma unroll
        for (int k = 0; k < NCONF; ++k) {
            double p[3];
            cfg.template load<B, spec::P_BJ[E], spec::P_DA[E], spec::P_DB[E], spec::P_DC[E]>(k, p);
            // J n_j + n_j x D, zero components dropped at compile time
            if constexpr (J != 0.0) { const double j = specc::P_J[E]; F[k][0] = fma(j, p[0], F[k][0]); F[k][1] = fma(j, p[1], F[k][1]); F[k][2] = fma(j, p[2], F[k][2]); }
            if constexpr (Dz != 0.0) { const double d = specc::P_DZ[E]; F[k][0] = fma(p[1], d, F[k][0]); F[k][1] = fma(p[0], -d, F[k][1]); }
            if constexpr (Dy != 0.0) { const double d = specc::P_DY[E]; F[k][0] = fma(p[2], -d, F[k][0]); F[k][2] = fma(p[0], d, F[k][2]); }
            if constexpr (Dx != 0.0) { const double d = specc::P_DX[E]; F[k][1] = fma(p[2], d, F[k][1]); F[k][2] = fma(p[1], -d, F[k][2]); }
        }
    });
    static_for<spec::QUAD_BEGIN[B], spec::QUAD_BEGIN[B + 1]>([&](auto e) {
        constexpr int E = decltype(e)::value;
#pragma unroll
        for (int k = 0; k < NCONF; ++k) {
            double P[3], Q[3], R[3];
            cfg.template load<B, spec::Q_B[E][0], spec::Q_D[E][0], spec::Q_D[E][1], spec::Q_D[E][2]>(k, P);
            cfg.template load<B, spec::Q_B[E][1], spec::Q_D[E][3], spec::Q_D[E][4], spec::Q_D[E][5]>(k, Q);
            cfg.template load<B, spec::Q_B[E][2], spec::Q_D[E][6], spec::Q_D[E][7], spec::Q_D[E][8]>(k, R);
            const double w = specc::Q_K[E] * fma(Q[0], R[0], fma(Q[1], R[1], Q[2] * R[2]));
            F[k][0] = fma(w, P[0], F[k][0]); F[k][1] = fma(w, P[1], F[k][1]); F[k][2] = fma(w, P[2], F[k][2]);
        }
    });
}

// (j^ . grad) n: central differences on the same sublattice, one-sided at open edges
template <int B, int NCONF, class Acc>
__device__ __forceinline__ void stt_gradient(const Acc &cfg, const Coord &c, const double (&own)[NCONF][3], double (&sg)[NCONF][3]) {
    static_for<0, 3>([&](auto dd) {
        constexpr int D = decltype(dd)::value;
        if constexpr (spec::STT_C[D] != 0.0) {
            constexpr int SA = D == 0 ? 1 : 0, SB = D == 1 ? 1 : 0, SC = D == 2 ? 1 : 0;
            constexpr bool PER = D == 0 ? spec::PER_A : (D == 1 ? spec::PER_B : spec::PER_C);
            constexpr int EXT = D == 0 ? spec::NA : (D == 1 ? spec::NB : spec::NC);
            const int x = D == 0 ? c.ia : (D == 1 ? c.ib : c.ic);
            const bool hp = PER || x + 1 < EXT, hm = PER || x > 0;
            const double w = specc::STT_C[D] * ((hp && hm) ? 0.5 : ((hp || hm) ? 1.0 : 0.0));
#pragma unroll
            for (int k = 0; k < NCONF; ++k) {
                double vp[3], vm[3];
                cfg.template load<B, B, SA, SB, SC>(k, vp); cfg.template load<B, B, -SA, -SB, -SC>(k, vm);
                if constexpr (!PER) {      // ghost cells of an open edge hold zeros: use the own spin for the one-sided difference
                    if (!hp) { vp[0] = own[k][0]; vp[1] = own[k][1]; vp[2] = own[k][2]; }
                    if (!hm) { vm[0] = own[k][0]; vm[1] = own[k][1]; vm[2] = own[k][2]; }
                }
                sg[k][0] = fma(w, vp[0] - vm[0], sg[k][0]); sg[k][1] = fma(w, vp[1] - vm[1], sg[k][1]); sg[k][2] = fma(w, vp[2] - vm[2], sg[k][2]);
            }
        }
    });
}

// A = pre [F + alpha n x F] + stt_s s + stt_x n x s   (Eq. 10 as dn/dt = n x A)
// ir: mu_b / mu_i of the site when per-site moments are set (the 1/mu_i of Eq. 10)
template <int B>
__device__ __forceinline__ void rotation_field(const double (&n)[3], const double (&F)[3], const double (&sg)[3], double (&A)[3], const double ir = 1.0) {
    const double pre = spec::HAS_SITE_MU ? specc::PRE[B] * ir : specc::PRE[B], pa = spec::HAS_SITE_MU ? specc::PREA[B] * ir : specc::PREA[B];
    const double cx = fma(n[1], F[2], -n[2] * F[1]), cy = fma(n[2], F[0], -n[0] * F[2]), cz = fma(n[0], F[1], -n[1] * F[0]);
    if constexpr (spec::DAMPING_ONLY) {      // :168 "only the damping part of the LLG equation": the solvers become minimisers
        A[0] = pa * cx; A[1] = pa * cy; A[2] = pa * cz;
    } else {
        A[0] = fma(pa, cx, pre * F[0]);
        A[1] = fma(pa, cy, pre * F[1]);
        A[2] = fma(pa, cz, pre * F[2]);
    }
    if constexpr (spec::STT_ON) {
        const double sx = fma(n[1], sg[2], -n[2] * sg[1]), sy = fma(n[2], sg[0], -n[0] * sg[2]), sz = fma(n[0], sg[1], -n[1] * sg[0]);
        A[0] += fma(specc::STT_X, sx, specc::STT_S * sg[0]);
        A[1] += fma(specc::STT_X, sy, specc::STT_S * sg[1]);
        A[2] += fma(specc::STT_X, sz, specc::STT_S * sg[2]);
    }
}

template <int B>
__device__ __forceinline__ bool locate(Coord &c, int &idx, int brick) {
    constexpr int nbx = (spec::NA + spec::BX - 1) / spec::BX, nby = (spec::NB + spec::BY - 1) / spec::BY;
    const int bx = brick % nbx;
    brick /= nbx;
    const int by = brick % nby, bz = brick / nby;
    const int t = threadIdx.x;
    c.ia = bx * spec::BX + (t % spec::BX);
    c.ib = by * spec::BY + (t / spec::BX) % spec::BY;
    c.ic = bz * spec::BZ + t / (spec::BX * spec::BY);
    idx = B * spec::SUB + (c.ic + spec::LC) * PLANE + (c.ib + spec::LB) * ROW + (c.ia + spec::LA);
    return (c.ia < spec::NA) && (c.ib < spec::NB) && (c.ic < spec::NC);
}

// image / sigma_scale: batched images draw independent noise, each at its own temperature (sigma ~ sqrt(T)); 0 / 1.0 otherwise
template <int B>
__device__ __forceinline__ void thermal_force(const Coord &c, u64 step, u32 seed_lo, u32 seed_hi, double (&f)[3], u32 image = 0u,
                                              double sigma_scale = 1.0) {
    if constexpr (spec::THERMAL_ON) {
        const u32 cell = (u32)(c.ia + spec::NA * c.ib + (spec::NA * spec::NB) * c.ic) + (u32)spec::CELL_OFF;      // the GLOBAL cell (slab decomposition)
        double xi[3];
        spin::thermal_xi(seed_lo, seed_hi, step, (u32)B + (u32)spec::NBASIS * cell, xi, image);
        const double sg = __dmul_rn(specc::SIGMA[B], sigma_scale);
        // rounded products (never contracted into a following add): the cached and the regenerated thermal field are the same bits
        f[0] = __dmul_rn(sg, xi[0]); f[1] = __dmul_rn(sg, xi[1]); f[2] = __dmul_rn(sg, xi[2]);
    } else {
        f[0] = -0.0; f[1] = -0.0; f[2] = -0.0;      // additive identity that the compiler may fold away (x + -0.0 == x exactly)
    }
}

// pinned spins: flags in boundary order b + NBASIS * cell; a pinned spin is copied, never updated
template <int B>
__device__ __forceinline__ bool is_pinned(const unsigned char *__restrict__ pin, const Coord &c) {
    if constexpr (spec::HAS_PIN) return pin[B + spec::NBASIS * (c.ia + spec::NA * (c.ib + spec::NB * c.ic))] != 0;
    else return false;
}

// per-site moments ("atoms of different types"): mu_i / mu_b in boundary order, like the pinning flags
template <int B>
__device__ __forceinline__ double site_ratio(const double *__restrict__ mur, const Coord &c) {
    if constexpr (spec::HAS_SITE_MU) return __ldg(mur + (B + spec::NBASIS * (c.ia + spec::NA * (c.ib + spec::NB * c.ic))));
    else return 1.0;
}

// Programmatic dependent launch (spec::PDL; the host then launches the sweep with programmatic stream serialisation): let the next
// kernel of the stream become resident as soon as every block of this one has started, and wait here -- before the first access to
// anything another kernel writes -- until the previous kernel has completed and its stores are visible.  Semantics of the stream
// order are unchanged; the launch latency and the block ramp of each sweep overlap the tail of the one before.
__device__ __forceinline__ void pdl_entry() {
    if constexpr (spec::PDL == 1) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if constexpr (spec::PDL != 0) asm volatile("griddepcontrol.wait;" ::: "memory");
}
__device__ __forceinline__ void pdl_exit() {
    if constexpr (spec::PDL == 2) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

template <int B, bool CG = false>
__device__ __forceinline__ void predictor_body(const double *__restrict__ n, const double *__restrict__ fddi, double *__restrict__ np,
                                               double *__restrict__ Aout, u64 step, u32 seed_lo, u32 seed_hi, const unsigned char *__restrict__ pin,
                                               const double *__restrict__ mur, int brick, u32 image = 0u, double sigma_scale = 1.0) {
    Coord c;
    int idx;
    if (!locate<B>(c, idx, brick)) return;
    GlobalAcc<1, CG> cfg;
    cfg.cfg[0] = n + idx;
    double own[1][3], F[1][3], sg[1][3] = {{0.0, 0.0, 0.0}};
    load3<0, CG>(cfg.cfg[0], own[0]);
    if (is_pinned<B>(pin, c)) { store_spin(np + idx, c, own[0]); return; }
    const double zr = site_ratio<B>(mur, c), ir = spec::HAS_SITE_MU ? 1.0 / zr : 1.0;
    if constexpr (spec::HAS_SITE_MU && spec::THERMAL_ON) sigma_scale *= sqrt(zr);      // sigma_i ~ sqrt(mu_i) (Eq. 11)
    thermal_force<B>(c, step, seed_lo, seed_hi, F[0], image, sigma_scale);
    // the thermal field of the step is the same in both sweeps (R11): generating it costs two Philox blocks, two logarithms and three
    // trigonometric evaluations per spin, so the predictor keeps it for the corrector (24 B/spin written and read back)
    if constexpr (spec::CACHE_NOISE) store3(Aout + idx, F[0]);
    force<B, 1>(cfg, own, F, zr);
    if constexpr (spec::HAS_DDI) { double d[3]; load3<0, CG>(fddi + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
    if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
    double A[3], out[3];
    rotation_field<B>(own[0], F[0], sg[0], A, ir);
    if constexpr (spec::SOLVER == 0) spin::rodrigues(A, specc::DT, specc::DT2, own[0], out);                 // B5
    else if constexpr (spec::SOLVER == 1) { out[0] = own[0][0]; out[1] = own[0][1]; out[2] = own[0][2]; spin::heun_add(own[0], A, specc::DT, out); }   // B3
    else spin::imp_update(A, specc::HDT, own[0], out);                                                        // C5
    store_spin(np + idx, c, out);
    if constexpr (spec::STORE_A) store3(Aout + idx, A);
}

template <int B, bool CG = false>
__device__ __forceinline__ void corrector_body(const double *__restrict__ n, const double *__restrict__ np, const double *__restrict__ fddi_n,
                                               const double *__restrict__ fddi_np, const double *__restrict__ Ain, double *__restrict__ nout,
                                               u64 step, u32 seed_lo, u32 seed_hi, const unsigned char *__restrict__ pin, const double *__restrict__ mur, int brick,
                                               u32 image = 0u, double sigma_scale = 1.0) {
    Coord c;
    int idx;
    if (!locate<B>(c, idx, brick)) return;
    double th[3], A[3], Ap[3], n0[3];
    load3<0, CG>(n + idx, n0);
    if (is_pinned<B>(pin, c)) { store_spin(nout + idx, c, n0); return; }
    const double zr = site_ratio<B>(mur, c), ir = spec::HAS_SITE_MU ? 1.0 / zr : 1.0;
    if constexpr (spec::HAS_SITE_MU && spec::THERMAL_ON) sigma_scale *= sqrt(zr);
    if constexpr (spec::CACHE_NOISE) load3<0, CG>(Ain + idx, th);
    else thermal_force<B>(c, step, seed_lo, seed_hi, th, image, sigma_scale);
    if constexpr (spec::SOLVER == 2) {
        // SIB corrector (C11): A at the midpoint configuration, the implicit-midpoint structure applied to n(t); A(n) is not needed
        const MidAcc<CG> cfg = {n + idx, np + idx};
        double own[1][3], F[1][3] = {{th[0], th[1], th[2]}}, sg[1][3] = {{0.0, 0.0, 0.0}};
        cfg.template load<B, B, 0, 0, 0>(0, own[0]);
        force<B, 1>(cfg, own, F, zr);
        if constexpr (spec::HAS_DDI) {      // the dipolar force is linear in the configuration: its value at the midpoint is the mean
            double d[3], e[3];
            load3<0, CG>(fddi_n + idx, d); load3<0, CG>(fddi_np + idx, e);
            F[0][0] += 0.5 * (d[0] + e[0]); F[0][1] += 0.5 * (d[1] + e[1]); F[0][2] += 0.5 * (d[2] + e[2]);
        }
        if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
        rotation_field<B>(own[0], F[0], sg[0], Ap, ir);
        double out[3];
        spin::imp_update(Ap, specc::HDT, n0, out);
        store_spin(nout + idx, c, out);
        return;
    }
    double np0[3] = {0.0, 0.0, 0.0};
    if constexpr (spec::STORE_A) {
        GlobalAcc<1, CG> cfg;
        cfg.cfg[0] = np + idx;
        double own[1][3], F[1][3] = {{th[0], th[1], th[2]}}, sg[1][3] = {{0.0, 0.0, 0.0}};
        load3<0, CG>(cfg.cfg[0], own[0]);
        force<B, 1>(cfg, own, F, zr);
        if constexpr (spec::HAS_DDI) { double d[3]; load3<0, CG>(fddi_np + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
        if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
        rotation_field<B>(own[0], F[0], sg[0], Ap, ir);
        load3<0, CG>(Ain + idx, A);
    } else if constexpr (spec::SPLIT_CORR) {
        // the two fields one after the other (fewer live registers, more resident warps) instead of interleaved
        {
            GlobalAcc<1, CG> cfg;
            cfg.cfg[0] = n + idx;
            double own[1][3] = {{n0[0], n0[1], n0[2]}}, F[1][3] = {{th[0], th[1], th[2]}}, sg[1][3] = {{0.0, 0.0, 0.0}};
            force<B, 1>(cfg, own, F, zr);
            if constexpr (spec::HAS_DDI) { double d[3]; load3<0, CG>(fddi_n + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
            if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
            rotation_field<B>(own[0], F[0], sg[0], A, ir);
        }
        {
            GlobalAcc<1, CG> cfg;
            cfg.cfg[0] = np + idx;
            double own[1][3], F[1][3] = {{th[0], th[1], th[2]}}, sg[1][3] = {{0.0, 0.0, 0.0}};
            load3<0, CG>(cfg.cfg[0], own[0]);
            np0[0] = own[0][0]; np0[1] = own[0][1]; np0[2] = own[0][2];
            force<B, 1>(cfg, own, F, zr);
            if constexpr (spec::HAS_DDI) { double d[3]; load3<0, CG>(fddi_np + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
            if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
            rotation_field<B>(own[0], F[0], sg[0], Ap, ir);
        }
    } else {
        GlobalAcc<2, CG> cfg;
        cfg.cfg[0] = n + idx; cfg.cfg[1] = np + idx;
        double own[2][3], F[2][3] = {{th[0], th[1], th[2]}, {th[0], th[1], th[2]}}, sg[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
        own[0][0] = n0[0]; own[0][1] = n0[1]; own[0][2] = n0[2];
        load3<0, CG>(cfg.cfg[1], own[1]);
        np0[0] = own[1][0]; np0[1] = own[1][1]; np0[2] = own[1][2];
        force<B, 2>(cfg, own, F, zr);
        if constexpr (spec::HAS_DDI) {
            double d[3];
            load3<0, CG>(fddi_n + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2];
            load3<0, CG>(fddi_np + idx, d); F[1][0] += d[0]; F[1][1] += d[1]; F[1][2] += d[2];
        }
        if constexpr (spec::STT_ON) stt_gradient<B, 2>(cfg, c, own, sg);
        rotation_field<B>(own[0], F[0], sg[0], A, ir);
        rotation_field<B>(own[1], F[1], sg[1], Ap, ir);
    }
    double out[3];
    if constexpr (spec::SOLVER == 1) {
        // Heun corrector (B4): n + dt/2 (n x A + n^p x A^p), renormalised every step
        out[0] = n0[0]; out[1] = n0[1]; out[2] = n0[2];
        spin::heun_add(n0, A, specc::HDT, out);
        spin::heun_add(np0, Ap, specc::HDT, out);
        spin::renormalise_general(out);
    } else {
        // A^c = (A + A^p)/2: the factor 1/2 is folded into the time step (dt/2, dt^2/4 are exact scalings, the result is bit-identical)
        const double Ac[3] = {A[0] + Ap[0], A[1] + Ap[1], A[2] + Ap[2]};
        spin::rodrigues(Ac, specc::HDT, specc::QDT2, n0, out);
        spin::renormalise(out);
    }
    store_spin(nout + idx, c, out);
}

// One stage of the classical 4th-order Runge-Kutta solver on dn/dt = f(n) = n x A(n):
//   k = f(y);  stage 0: acc = k, y' = n + dt/2 k;  1: acc += 2k, y' = n + dt/2 k;  2: acc += 2k, y' = n + dt k;
//   stage 3: n(t+dt) = n + dt/6 (acc + k), renormalised.  Stage configurations are not renormalised; one thermal field per step.
template <int B>
__device__ __forceinline__ void rk4_stage_body(const double *__restrict__ base, const double *__restrict__ y, double *__restrict__ ynext,
                                               double *__restrict__ acc, double *__restrict__ noise, const double *__restrict__ fddi, int stage,
                                               u64 step, u32 seed_lo, u32 seed_hi, const unsigned char *__restrict__ pin, const double *__restrict__ mur,
                                               int brick) {
    Coord c;
    int idx;
    if (!locate<B>(c, idx, brick)) return;
    double n0[3];
    load3<0>(base + idx, n0);
    if (is_pinned<B>(pin, c)) { store_spin(ynext + idx, c, n0); return; }
    const double zr = site_ratio<B>(mur, c), ir = spec::HAS_SITE_MU ? 1.0 / zr : 1.0;
    const double sscale = (spec::HAS_SITE_MU && spec::THERMAL_ON) ? sqrt(zr) : 1.0;
    GlobalAcc<1> cfg;
    cfg.cfg[0] = y + idx;
    double own[1][3], F[1][3], sg[1][3] = {{0.0, 0.0, 0.0}};
    load3<0>(cfg.cfg[0], own[0]);
    if constexpr (spec::THERMAL_ON && !spec::HAS_DDI) {      // generated once per step, kept for the other three stages
        if (stage == 0) { thermal_force<B>(c, step, seed_lo, seed_hi, F[0], 0u, sscale); store3(noise + idx, F[0]); }
        else load3<0>(noise + idx, F[0]);
    } else {
        thermal_force<B>(c, step, seed_lo, seed_hi, F[0], 0u, sscale);
    }
    force<B, 1>(cfg, own, F, zr);
    if constexpr (spec::HAS_DDI) { double d[3]; load3<0>(fddi + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
    if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
    double A[3], k[3] = {0.0, 0.0, 0.0};
    rotation_field<B>(own[0], F[0], sg[0], A, ir);
    spin::heun_add(own[0], A, 1.0, k);                      // k = y x A
    double a[3] = {0.0, 0.0, 0.0};
    if (stage > 0) load3<0>(acc + idx, a);
    double out[3];
    if (stage < 3) {
        const double w = stage == 0 ? 1.0 : 2.0, h = stage == 2 ? specc::DT : specc::HDT;
        a[0] = fma(w, k[0], a[0]); a[1] = fma(w, k[1], a[1]); a[2] = fma(w, k[2], a[2]);
        store3(acc + idx, a);
        out[0] = fma(h, k[0], n0[0]); out[1] = fma(h, k[1], n0[1]); out[2] = fma(h, k[2], n0[2]);
    } else {
        const double h = specc::DT / 6.0;
        out[0] = fma(h, a[0] + k[0], n0[0]); out[1] = fma(h, a[1] + k[1], n0[1]); out[2] = fma(h, a[2] + k[2], n0[2]);
        spin::renormalise_general(out);
    }
    store_spin(ynext + idx, c, out);
}

template <int B, class Fn>
__device__ __forceinline__ void dispatch_basis(int b, Fn &&fn) {
    if constexpr (B < spec::NBASIS) {
        if (b == B) fn(Int<B>{});
        else dispatch_basis<B + 1>(b, fn);
    }
}

}  // namespace spinjit

extern "C" __global__ void SPIN_BOUNDS(spec::BX *spec::BY *spec::BZ)
    jit_predictor(const double *__restrict__ n, const double *__restrict__ fddi, double *__restrict__ np, double *__restrict__ Aout,
                  const unsigned long long *__restrict__ d_step, unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi,
                  const unsigned char *__restrict__ pin, const double *__restrict__ img_sigma, const double *__restrict__ mu_ratio,
                  unsigned int brick0) {
    spinjit::pdl_entry();
    const unsigned long long step = *d_step + step_add;
    // batched images: blockIdx.z selects the image; every per-spin array holds the images one after the other
    const unsigned int image = spec::MULTI_IMAGE ? blockIdx.z : 0u;
    const size_t off = spec::MULTI_IMAGE ? (size_t)image * ((size_t)spec::NBASIS * spec::SUB) : (size_t)0;
    const double scale = (spec::MULTI_IMAGE && img_sigma) ? img_sigma[image] : 1.0;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        spinjit::predictor_body<decltype(b)::value>(n + off, fddi + off, np + off, Aout + off, step, seed_lo, seed_hi, pin, mu_ratio, (int)(brick0 + blockIdx.x), image, scale);
    });
    spinjit::pdl_exit();
}

extern "C" __global__ void SPIN_BOUNDS(spec::BX *spec::BY *spec::BZ)
    jit_corrector(const double *__restrict__ n, const double *__restrict__ np, const double *__restrict__ fddi_n,
                  const double *__restrict__ fddi_np, const double *__restrict__ Ain, double *__restrict__ nout,
                  const unsigned long long *__restrict__ d_step, unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi,
                  const unsigned char *__restrict__ pin, const double *__restrict__ img_sigma, const double *__restrict__ mu_ratio,
                  unsigned int brick0) {
    spinjit::pdl_entry();
    const unsigned long long step = *d_step + step_add;
    const unsigned int image = spec::MULTI_IMAGE ? blockIdx.z : 0u;
    const size_t off = spec::MULTI_IMAGE ? (size_t)image * ((size_t)spec::NBASIS * spec::SUB) : (size_t)0;
    const double scale = (spec::MULTI_IMAGE && img_sigma) ? img_sigma[image] : 1.0;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        // The corrector walks the bricks in the opposite order to the predictor: what the predictor touched last (the tail of n and of
        // n^p) is still in the 126 MB L2 and is read first; it ends at brick 0, where the next predictor starts.
        const int brick = (int)brick0 + (spec::REVERSE_CORR ? (int)(gridDim.x - 1u - blockIdx.x) : (int)blockIdx.x);      // brick0: first brick of a range launch
        spinjit::corrector_body<decltype(b)::value>(n + off, np + off, fddi_n + off, fddi_np + off, Ain + off, nout + off, step, seed_lo, seed_hi, pin,
                                                    mu_ratio, brick, image, scale);
    });
    spinjit::pdl_exit();
}

extern "C" __global__ void SPIN_BOUNDS(spec::BX *spec::BY *spec::BZ)
    jit_rk4_stage(const double *__restrict__ base, const double *__restrict__ y, double *__restrict__ ynext, double *__restrict__ acc,
                  double *__restrict__ noise, const double *__restrict__ fddi, int stage, const unsigned long long *__restrict__ d_step,
                  unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi, const unsigned char *__restrict__ pin,
                  const double *__restrict__ mu_ratio) {
    const unsigned long long step = *d_step + step_add;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        spinjit::rk4_stage_body<decltype(b)::value>(base, y, ynext, acc, noise, fddi, stage, step, seed_lo, seed_hi, pin, mu_ratio, (int)blockIdx.x);
    });
}

// ---------------------------------------------------------------------------------------------------------------------------
// Launch-bound lattices ("limited by the overhead of CUDA kernel launches"): ALL steps of an llg_iterate call in ONE
// cooperative launch.  Every block walks its share of the bricks, predictor sweep -> grid barrier -> corrector sweep -> grid
// barrier, ping-ponging between the two n buffers; the arrays are read with coherent loads (not the read-only path) because other blocks
// rewrite them between barriers.  The barrier is a monotone arrival counter in global memory (release: fence + atomic add; acquire: polling
// load + fence); a lost arrival traps instead of hanging the device.  All blocks are co-resident (cooperative launch).
namespace spinjit {
__device__ __forceinline__ void grid_barrier(unsigned int *bar, unsigned int nblocks, unsigned int &target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        target += nblocks;
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned int seen = 0, polls = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
            if (++polls > (1u << 28)) __trap();
        } while (seen < target);
        __threadfence();
    }
    __syncthreads();
}
}  // namespace spinjit

namespace spinjit {
// hardware barrier of a thread-block cluster: every thread of every block arrives (release) and waits (acquire); cluster scope orders
// the global-memory traffic of the blocks just like the grid barrier above, at a fraction of its latency
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <class Barrier>
__device__ __forceinline__ void all_steps(double *__restrict__ n0, double *__restrict__ n1, double *__restrict__ np, double *__restrict__ aux,
                                          u64 step0, unsigned int nsteps, u32 seed_lo, u32 seed_hi, const unsigned char *__restrict__ pin,
                                          const double *__restrict__ mur, Barrier &&barrier) {
    constexpr int NBRICKS = ((spec::NA + spec::BX - 1) / spec::BX) * ((spec::NB + spec::BY - 1) / spec::BY) * ((spec::NC + spec::BZ - 1) / spec::BZ);
    for (unsigned int k = 0; k < nsteps; ++k) {
        const double *n = (k & 1u) ? n1 : n0;
        double *nout = (k & 1u) ? n0 : n1;
        const u64 step = step0 + k;
        for (int item = blockIdx.x; item < NBRICKS * spec::NBASIS; item += gridDim.x)
            dispatch_basis<0>(item / NBRICKS, [&](auto b) {
                predictor_body<decltype(b)::value, true>(n, nullptr, np, aux, step, seed_lo, seed_hi, pin, mur, item % NBRICKS);
            });
        barrier();
        for (int item = blockIdx.x; item < NBRICKS * spec::NBASIS; item += gridDim.x)
            dispatch_basis<0>(item / NBRICKS, [&](auto b) {
                corrector_body<decltype(b)::value, true>(n, np, nullptr, nullptr, aux, nout, step, seed_lo, seed_hi, pin, mur, item % NBRICKS);
            });
        barrier();
    }
}
}  // namespace spinjit

extern "C" __global__ void SPIN_BOUNDS(spec::BX *spec::BY *spec::BZ)
    jit_steps_coop(double *__restrict__ n0, double *__restrict__ n1, double *__restrict__ np, double *__restrict__ aux,
                   const unsigned long long *__restrict__ d_step, unsigned int nsteps, unsigned int seed_lo, unsigned int seed_hi,
                   const unsigned char *__restrict__ pin, unsigned int *bar, const double *__restrict__ mu_ratio) {
    unsigned int target = 0;
    spinjit::all_steps(n0, n1, np, aux, *d_step, nsteps, seed_lo, seed_hi, pin, mu_ratio, [&]() { spinjit::grid_barrier(bar, gridDim.x, target); });
}

// the same for lattices of at most 16 bricks: the whole grid is ONE thread-block cluster and the barrier is the cluster's hardware barrier
extern "C" __global__ void SPIN_BOUNDS(spec::BX *spec::BY *spec::BZ)
    jit_steps_cluster(double *__restrict__ n0, double *__restrict__ n1, double *__restrict__ np, double *__restrict__ aux,
                      const unsigned long long *__restrict__ d_step, unsigned int nsteps, unsigned int seed_lo, unsigned int seed_hi,
                      const unsigned char *__restrict__ pin, const double *__restrict__ mu_ratio) {
    spinjit::all_steps(n0, n1, np, aux, *d_step, nsteps, seed_lo, seed_hi, pin, mu_ratio, []() { spinjit::cluster_barrier(); });
}

#ifdef SPIN_MARCH
#include "spin_jit_march.cuh"
#endif
