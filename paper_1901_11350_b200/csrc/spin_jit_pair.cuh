// spin_jit_pair.cuh -- the two Depondt sweeps with TWO sites per thread and 128-bit accesses (included by spin_jit_kernels.cuh when
// SPIN_PAIR is defined).
//
// Why (profiles/r1c_README.md, r1e): the brick kernels are bound by the L1 data pipe.  Of the 7 vector loads per configuration of a
// nearest-neighbour stencil, the three along a (x-1, x, x+1) fetch nearly the same 256 bytes per warp three times, and the two
// unaligned ones cost three wavefronts instead of two.  Here a thread owns the sites (ia, ia+1), ia even: every partner comes from an
// aligned double2 {even site, odd site}, and the loads that both sites issue for the same double2 are one instruction (identical
// read-only loads are merged by the compiler).  Along a the pair needs the double2 at -2, 0, +2 (3 x 4 wavefronts per 64 sites instead
// of 2 x (2 + 3 + 3)); along b and c one double2 per partner replaces two scalar loads (same wavefronts, half the instructions); the
// results leave as double2 stores.  Two independent dependency chains per thread also hide more latency per resident warp.
// Arithmetic, gather table, ghost images, noise: the code of the brick kernels (force<>, rotation_field<>, rodrigues), so the result is
// bit-identical.
//
// Needs spec::NA even and an even ghost offset (all of SUB, PLANE, ROW, LA even: every double2 is 16-byte aligned); spec must define
// VBX (even), VBY, VBZ: the brick of sites per block; threads per block = VBX/2 * VBY * VBZ.
#pragma once

namespace spinpair {
using namespace spinjit;

static_assert(spec::NA % 2 == 0 && spec::LA % 2 == 0 && spec::PA % 2 == 0 && spec::SUB % 2 == 0 && spec::VBX % 2 == 0, "pair sweeps need even rows");

constexpr int HBX = spec::VBX / 2;
constexpr int NTHREADS = HBX * spec::VBY * spec::VBZ;
constexpr int NBX = (spec::NA + spec::VBX - 1) / spec::VBX, NBY = (spec::NB + spec::VBY - 1) / spec::VBY, NBZ = (spec::NC + spec::VBZ - 1) / spec::VBZ;

__device__ __forceinline__ double2 ldg2(const double *q) { return __ldg(reinterpret_cast<const double2 *>(q)); }

// S = 0: the even site of the pair, S = 1: the odd one.  cfg[k] points at the x component of the EVEN site in configuration k.
template <int NCONF, int S>
struct PairAcc {
    const double *cfg[NCONF];
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int k, double (&v)[3]) const {
        constexpr int e = S + DA;                                           // position along a relative to the even site
        constexpr int p = (e >= 0 ? e / 2 : -((1 - e) / 2)) * 2;            // the double2 that holds it starts here (floor to even)
        constexpr bool hi = (e - p) != 0;
        constexpr int O = lin<B, BJ, 0, DB, DC>() + p;
        const double2 x = ldg2(cfg[k] + O), y = ldg2(cfg[k] + O + spec::PA), z = ldg2(cfg[k] + O + 2 * spec::PA);
        v[0] = hi ? x.y : x.x; v[1] = hi ? y.y : y.x; v[2] = hi ? z.y : z.x;
    }
};

__device__ __forceinline__ void load_pair(const double *q, double (&a)[3], double (&b)[3]) {
    const double2 x = ldg2(q), y = ldg2(q + spec::PA), z = ldg2(q + 2 * spec::PA);
    a[0] = x.x; a[1] = y.x; a[2] = z.x;
    b[0] = x.y; b[1] = y.y; b[2] = z.y;
}

// both spins with one 128-bit store per component, then the periodic images of each (edge sites only)
__device__ __forceinline__ void store_pair(double *__restrict__ q, const Coord &c0, const double (&a)[3], const double (&b)[3]) {
    *reinterpret_cast<double2 *>(q) = make_double2(a[0], b[0]);
    *reinterpret_cast<double2 *>(q + spec::PA) = make_double2(a[1], b[1]);
    *reinterpret_cast<double2 *>(q + 2 * spec::PA) = make_double2(a[2], b[2]);
    Coord c1 = c0;
    c1.ia += 1;
    store_images(q, c0, a);
    store_images(q + 1, c1, b);
}

// the even site of this thread's pair; false if outside the lattice
template <int B>
__device__ __forceinline__ bool locate_pair(Coord &c, int &idx, int brick) {
    const int bx = brick % NBX;
    brick /= NBX;
    const int by = brick % NBY, bz = brick / NBY;
    const int t = threadIdx.x;
    c.ia = bx * spec::VBX + 2 * (t % HBX);
    c.ib = by * spec::VBY + (t / HBX) % spec::VBY;
    c.ic = bz * spec::VBZ + t / (HBX * spec::VBY);
    idx = B * spec::SUB + (c.ic + spec::LC) * PLANE + (c.ib + spec::LB) * ROW + (c.ia + spec::LA);
    return (c.ia < spec::NA) && (c.ib < spec::NB) && (c.ic < spec::NC);
}

template <int B>
__device__ __forceinline__ void predictor_pair(const double *__restrict__ n, const double *__restrict__ fddi, double *__restrict__ np,
                                               u64 step, u32 seed_lo, u32 seed_hi, int brick) {
    Coord c0;
    int idx;
    if (!locate_pair<B>(c0, idx, brick)) return;
    Coord c1 = c0;
    c1.ia += 1;
    PairAcc<1, 0> a0;
    PairAcc<1, 1> a1;
    a0.cfg[0] = n + idx;
    a1.cfg[0] = n + idx;
    double own0[1][3], own1[1][3], F0[1][3], F1[1][3], sg0[1][3] = {{0.0, 0.0, 0.0}}, sg1[1][3] = {{0.0, 0.0, 0.0}};
    load_pair(n + idx, own0[0], own1[0]);
    thermal_force<B>(c0, step, seed_lo, seed_hi, F0[0]);
    thermal_force<B>(c1, step, seed_lo, seed_hi, F1[0]);
    force<B, 1>(a0, own0, F0);
    force<B, 1>(a1, own1, F1);
    if constexpr (spec::HAS_DDI) {
        double d0[3], d1[3];
        load_pair(fddi + idx, d0, d1);
        F0[0][0] += d0[0]; F0[0][1] += d0[1]; F0[0][2] += d0[2];
        F1[0][0] += d1[0]; F1[0][1] += d1[1]; F1[0][2] += d1[2];
    }
    if constexpr (spec::STT_ON) { stt_gradient<B, 1>(a0, c0, own0, sg0); stt_gradient<B, 1>(a1, c1, own1, sg1); }
    double A0[3], A1[3], out0[3], out1[3];
    rotation_field<B>(own0[0], F0[0], sg0[0], A0);
    rotation_field<B>(own1[0], F1[0], sg1[0], A1);
    spin::rodrigues(A0, specc::DT, specc::DT2, own0[0], out0);
    spin::rodrigues(A1, specc::DT, specc::DT2, own1[0], out1);
    store_pair(np + idx, c0, out0, out1);
}

// one site of the pair in the corrector: both fields interleaved (as the brick corrector); returns A + A^p (the 1/2 is folded into dt)
template <int B, int S>
__device__ __forceinline__ void corrector_field(const double *__restrict__ n, const double *__restrict__ np, const Coord &c, const double (&th)[3],
                                                const double (&n0)[3], const double (&np0)[3], const double (&dn)[3], const double (&dnp)[3],
                                                double (&Ac)[3]) {
    PairAcc<2, S> acc;
    acc.cfg[0] = n;
    acc.cfg[1] = np;
    double A[3], Ap[3];
    double own[2][3] = {{n0[0], n0[1], n0[2]}, {np0[0], np0[1], np0[2]}};
    double F[2][3] = {{th[0], th[1], th[2]}, {th[0], th[1], th[2]}}, sg[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
    force<B, 2>(acc, own, F);
    if constexpr (spec::HAS_DDI) {
        F[0][0] += dn[0]; F[0][1] += dn[1]; F[0][2] += dn[2];
        F[1][0] += dnp[0]; F[1][1] += dnp[1]; F[1][2] += dnp[2];
    }
    if constexpr (spec::STT_ON) stt_gradient<B, 2>(acc, c, own, sg);
    rotation_field<B>(own[0], F[0], sg[0], A);
    rotation_field<B>(own[1], F[1], sg[1], Ap);
    Ac[0] = A[0] + Ap[0]; Ac[1] = A[1] + Ap[1]; Ac[2] = A[2] + Ap[2];
}

template <int B>
__device__ __forceinline__ void corrector_pair(const double *__restrict__ n, const double *__restrict__ np, const double *__restrict__ fddi_n,
                                               const double *__restrict__ fddi_np, double *__restrict__ nout, u64 step, u32 seed_lo, u32 seed_hi,
                                               int brick) {
    Coord c0;
    int idx;
    if (!locate_pair<B>(c0, idx, brick)) return;
    Coord c1 = c0;
    c1.ia += 1;
    double n0[3], n1[3], p0[3], p1[3], dn0[3] = {0.0, 0.0, 0.0}, dn1[3] = {0.0, 0.0, 0.0}, dp0[3] = {0.0, 0.0, 0.0}, dp1[3] = {0.0, 0.0, 0.0};
    double th0[3], th1[3];
    // the noise first (its slow paths use local memory), then all loads of both sites with nothing in between that could write
    // memory: the loads the two sites share are merged
    thermal_force<B>(c0, step, seed_lo, seed_hi, th0);
    thermal_force<B>(c1, step, seed_lo, seed_hi, th1);
    load_pair(n + idx, n0, n1);
    load_pair(np + idx, p0, p1);
    if constexpr (spec::HAS_DDI) { load_pair(fddi_n + idx, dn0, dn1); load_pair(fddi_np + idx, dp0, dp1); }
    double Ac0[3], Ac1[3], out0[3], out1[3];
    if constexpr (spec::SPLIT_CORR) {
        // the fields of n, then the fields of n^p (fewer live registers), each for both sites
        double sg0[1][3] = {{0.0, 0.0, 0.0}}, sg1[1][3] = {{0.0, 0.0, 0.0}}, A0[3], A1[3];
        PairAcc<1, 0> a0;
        PairAcc<1, 1> a1;
        {
            a0.cfg[0] = n + idx; a1.cfg[0] = n + idx;
            double own0[1][3] = {{n0[0], n0[1], n0[2]}}, own1[1][3] = {{n1[0], n1[1], n1[2]}};
            double F0[1][3] = {{th0[0], th0[1], th0[2]}}, F1[1][3] = {{th1[0], th1[1], th1[2]}};
            force<B, 1>(a0, own0, F0);
            force<B, 1>(a1, own1, F1);
            if constexpr (spec::HAS_DDI) {
                F0[0][0] += dn0[0]; F0[0][1] += dn0[1]; F0[0][2] += dn0[2];
                F1[0][0] += dn1[0]; F1[0][1] += dn1[1]; F1[0][2] += dn1[2];
            }
            if constexpr (spec::STT_ON) { stt_gradient<B, 1>(a0, c0, own0, sg0); stt_gradient<B, 1>(a1, c1, own1, sg1); }
            rotation_field<B>(own0[0], F0[0], sg0[0], A0);
            rotation_field<B>(own1[0], F1[0], sg1[0], A1);
        }
        {
            a0.cfg[0] = np + idx; a1.cfg[0] = np + idx;
            double own0[1][3] = {{p0[0], p0[1], p0[2]}}, own1[1][3] = {{p1[0], p1[1], p1[2]}};
            double F0[1][3] = {{th0[0], th0[1], th0[2]}}, F1[1][3] = {{th1[0], th1[1], th1[2]}};
            sg0[0][0] = sg0[0][1] = sg0[0][2] = 0.0; sg1[0][0] = sg1[0][1] = sg1[0][2] = 0.0;
            force<B, 1>(a0, own0, F0);
            force<B, 1>(a1, own1, F1);
            if constexpr (spec::HAS_DDI) {
                F0[0][0] += dp0[0]; F0[0][1] += dp0[1]; F0[0][2] += dp0[2];
                F1[0][0] += dp1[0]; F1[0][1] += dp1[1]; F1[0][2] += dp1[2];
            }
            if constexpr (spec::STT_ON) { stt_gradient<B, 1>(a0, c0, own0, sg0); stt_gradient<B, 1>(a1, c1, own1, sg1); }
            rotation_field<B>(own0[0], F0[0], sg0[0], Ac0);
            rotation_field<B>(own1[0], F1[0], sg1[0], Ac1);
        }
        Ac0[0] += A0[0]; Ac0[1] += A0[1]; Ac0[2] += A0[2];
        Ac1[0] += A1[0]; Ac1[1] += A1[1]; Ac1[2] += A1[2];
    } else {
        corrector_field<B, 0>(n + idx, np + idx, c0, th0, n0, p0, dn0, dp0, Ac0);
        corrector_field<B, 1>(n + idx, np + idx, c1, th1, n1, p1, dn1, dp1, Ac1);
    }
    spin::rodrigues(Ac0, specc::HDT, specc::QDT2, n0, out0);
    spin::renormalise(out0);
    spin::rodrigues(Ac1, specc::HDT, specc::QDT2, n1, out1);
    spin::renormalise(out1);
    store_pair(nout + idx, c0, out0, out1);
}

}  // namespace spinpair

extern "C" __global__ void SPIN_BOUNDS(spinpair::NTHREADS)
    jit_predictor_pair(const double *__restrict__ n, const double *__restrict__ fddi, double *__restrict__ np,
                       const unsigned long long *__restrict__ d_step, unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi) {
    const unsigned long long step = *d_step + step_add;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        spinpair::predictor_pair<decltype(b)::value>(n, fddi, np, step, seed_lo, seed_hi, (int)blockIdx.x);
    });
}

extern "C" __global__ void SPIN_BOUNDS(spinpair::NTHREADS)
    jit_corrector_pair(const double *__restrict__ n, const double *__restrict__ np, const double *__restrict__ fddi_n,
                       const double *__restrict__ fddi_np, double *__restrict__ nout, const unsigned long long *__restrict__ d_step,
                       unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi) {
    const unsigned long long step = *d_step + step_add;
    // bricks in reverse order, as jit_corrector: what the predictor wrote last is read first, while it is still in L2
    const int brick = spec::REVERSE_CORR ? (int)(gridDim.x - 1u - blockIdx.x) : (int)blockIdx.x;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        spinpair::corrector_pair<decltype(b)::value>(n, np, fddi_n, fddi_np, nout, step, seed_lo, seed_hi, brick);
    });
}
