// spin_kernels.cuh -- device code of the LLG hot path (sm_100a, fp64).
//
// One thread per spin; each spin GATHERS its own pair / quadruplet contributions (no atomics).  Thread blocks
// map to 3-D bricks of one sublattice so that the neighbours of a brick stay in L1/L2.  Interaction tables
// travel as a __grid_constant__ kernel parameter (constant bank), periodic-image index arithmetic is done
// in registers and skipped entirely for bricks that touch no boundary.
//
// Formulas (PAPER.md line numbers):
//   force      F_i = -dH/dn_i of Eq. 1 (:61-67) and Eq. 2 (:75), ":155 B_eff = -dH/dn_i"
//   LLG        Eq. 10 (:147-153) written as dn/dt = n x A (B1, :349)
//   noise      Eq. 11 (:157) scaled by 1/sqrt(dt) (:160), Philox4x32-10 keyed by (seed; spin, block, step)
//   Depondt    predictor n^p = R(A) n (B5 :371); A^c = (A + A^p)/2 (B6 :375); n <- R(A^c) n(t) (B7 :380)
#pragma once

#include "spinllg_internal.h"
#include "spin_device_math.cuh"

namespace spin {

struct Site {
    int ia, ib, ic, b;
    int idx;          // internal SoA index  b*Ncell + cell
    bool valid;
    bool interior;    // the whole brick is at least `reach` away from every boundary
};

template <int BX, int BY, int BZ>
__device__ __forceinline__ Site locate(const DevicePlan &P) {
    Site s;
    const int nbx = (P.Na + BX - 1) / BX, nby = (P.Nb + BY - 1) / BY;
    int brick = blockIdx.x;
    const int bx = brick % nbx;
    brick /= nbx;
    const int by = brick % nby, bz = brick / nby;
    const int t = threadIdx.x;
    const int x0 = bx * BX, y0 = by * BY, z0 = bz * BZ;
    s.ia = x0 + (t % BX);
    s.ib = y0 + (t / BX) % BY;
    s.ic = z0 + t / (BX * BY);
    s.b = blockIdx.y;
    s.valid = (s.ia < P.Na) && (s.ib < P.Nb) && (s.ic < P.Nc);
    s.idx = s.b * P.Ncell + s.ia + P.Na * (s.ib + P.Nb * s.ic);
    s.interior = (x0 >= P.reach[0]) && (x0 + BX + P.reach[0] <= P.Na) && (y0 >= P.reach[1]) &&
                 (y0 + BY + P.reach[1] <= P.Nb) && (z0 >= P.reach[2]) && (z0 + BZ + P.reach[2] <= P.Nc);
    return s;
}

// partner index with boundary conditions; returns false when the partner falls off an open edge
__device__ __forceinline__ bool partner(const DevicePlan &P, const Site &s, int da, int db, int dc, int bj, int lin,
                                        int &idx) {
    if (s.interior) {
        idx = s.idx + lin;
        return true;
    }
    int ja = s.ia + da, jb = s.ib + db, jc = s.ic + dc;
    bool ok = true;
    if (ja < 0) { ja += P.Na; ok = ok && P.perA; } else if (ja >= P.Na) { ja -= P.Na; ok = ok && P.perA; }
    if (jb < 0) { jb += P.Nb; ok = ok && P.perB; } else if (jb >= P.Nb) { jb -= P.Nb; ok = ok && P.perB; }
    if (jc < 0) { jc += P.Nc; ok = ok && P.perC; } else if (jc >= P.Nc) { jc -= P.Nc; ok = ok && P.perC; }
    idx = ok ? bj * P.Ncell + ja + P.Na * (jb + P.Nb * jc) : s.idx;
    return ok;
}

// ---------------------------------------------------------------------------------------------------------
// Short-range force of NCONF configurations that share the lattice (n and n^p in the corrector): the partner
// index is computed once per table entry and used for every configuration.
// cfg[c] points at the x component; y and z follow at +stride, +2*stride.
template <int NCONF>
__device__ __forceinline__ void short_range_force(const DevicePlan &P, const double *const (&cfg)[NCONF], const Site &s,
                                                  const double (&own)[NCONF][3], int mask, double (&F)[NCONF][3]) {
    const int b = s.b, st = P.stride;
    if (mask & T_ZEE) {
#pragma unroll
        for (int c = 0; c < NCONF; ++c) { F[c][0] += P.zee[b][0]; F[c][1] += P.zee[b][1]; F[c][2] += P.zee[b][2]; }
    }
    if ((mask & T_ANI) && P.K2[b] != 0.0) {
        const double kx = P.Kax[b][0], ky = P.Kax[b][1], kz = P.Kax[b][2], k2 = P.K2[b];
#pragma unroll
        for (int c = 0; c < NCONF; ++c) {
            const double p = k2 * (kx * own[c][0] + ky * own[c][1] + kz * own[c][2]);
            F[c][0] += p * kx; F[c][1] += p * ky; F[c][2] += p * kz;
        }
    }
    if (mask & (T_EXC | T_DMI)) {
        const double wj = (mask & T_EXC) ? 1.0 : 0.0, wd = (mask & T_DMI) ? 1.0 : 0.0;
        const bool all = (mask & T_EXC) && (mask & T_DMI);
        for (int e = P.pair_begin[b]; e < P.pair_begin[b + 1]; ++e) {
            const PairEntry &pe = P.pairs[e];
            int j;
            if (!partner(P, s, pe.da, pe.db, pe.dc, pe.bj, pe.lin, j)) continue;
            const double J = all ? pe.J : wj * pe.J;
            const double Dx = all ? pe.Dx : wd * pe.Dx, Dy = all ? pe.Dy : wd * pe.Dy, Dz = all ? pe.Dz : wd * pe.Dz;
#pragma unroll
            for (int c = 0; c < NCONF; ++c) {
                const double px = __ldg(cfg[c] + j), py = __ldg(cfg[c] + st + j), pz = __ldg(cfg[c] + 2 * st + j);
                // J n_j + n_j x D
                F[c][0] += J * px + (py * Dz - pz * Dy);
                F[c][1] += J * py + (pz * Dx - px * Dz);
                F[c][2] += J * pz + (px * Dy - py * Dx);
            }
        }
    }
    if (mask & T_QUAD) {
        for (int e = P.quad_begin[b]; e < P.quad_begin[b + 1]; ++e) {
            const QuadEntry &q = P.quads[e];
            int jp, jq, jr;
            bool ok = partner(P, s, q.d[0][0], q.d[0][1], q.d[0][2], q.b[0], q.lin[0], jp);
            ok = partner(P, s, q.d[1][0], q.d[1][1], q.d[1][2], q.b[1], q.lin[1], jq) && ok;
            ok = partner(P, s, q.d[2][0], q.d[2][1], q.d[2][2], q.b[2], q.lin[2], jr) && ok;
            if (!ok) continue;
#pragma unroll
            for (int c = 0; c < NCONF; ++c) {
                const double *x = cfg[c], *y = cfg[c] + st, *z = cfg[c] + 2 * st;
                const double w = q.K * (__ldg(x + jq) * __ldg(x + jr) + __ldg(y + jq) * __ldg(y + jr) + __ldg(z + jq) * __ldg(z + jr));
                F[c][0] += w * __ldg(x + jp); F[c][1] += w * __ldg(y + jp); F[c][2] += w * __ldg(z + jp);
            }
        }
    }
}

// (j^ . grad) n by central lattice differences on the same sublattice, one-sided at open edges (R14)
template <int NCONF>
__device__ __forceinline__ void stt_gradient(const DevicePlan &P, const double *const (&cfg)[NCONF], const Site &s,
                                             const double (&own)[NCONF][3], double (&sg)[NCONF][3]) {
    const int st = P.stride;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double cd = P.stt_c[d];
        if (cd == 0.0) continue;
        int jp, jm;
        const bool hp = partner(P, s, d == 0, d == 1, d == 2, s.b, d == 0 ? 1 : (d == 1 ? P.Na : P.Na * P.Nb), jp);
        const bool hm = partner(P, s, -(d == 0), -(d == 1), -(d == 2), s.b, d == 0 ? -1 : (d == 1 ? -P.Na : -P.Na * P.Nb), jm);
        const double w = cd * ((hp && hm) ? 0.5 : ((hp || hm) ? 1.0 : 0.0));
#pragma unroll
        for (int c = 0; c < NCONF; ++c) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double vp = hp ? __ldg(cfg[c] + k * st + jp) : own[c][k];
                const double vm = hm ? __ldg(cfg[c] + k * st + jm) : own[c][k];
                sg[c][k] += w * (vp - vm);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Eq. 10 as dn/dt = n x A:  A = pre [F + alpha n x F] + stt_s s + stt_x n x s
__device__ __forceinline__ void rotation_field(const DevicePlan &P, int b, const double (&n)[3], const double (&F)[3],
                                               const double (&sg)[3], double (&A)[3]) {
    const double pre = P.pre[b], al = P.alpha;
    const double cx = n[1] * F[2] - n[2] * F[1], cy = n[2] * F[0] - n[0] * F[2], cz = n[0] * F[1] - n[1] * F[0];
    A[0] = pre * (F[0] + al * cx);
    A[1] = pre * (F[1] + al * cy);
    A[2] = pre * (F[2] + al * cz);
    if (P.stt_on) {
        const double sx = n[1] * sg[2] - n[2] * sg[1], sy = n[2] * sg[0] - n[0] * sg[2], sz = n[0] * sg[1] - n[1] * sg[0];
        A[0] += P.stt_s * sg[0] + P.stt_x * sx;
        A[1] += P.stt_s * sg[1] + P.stt_x * sy;
        A[2] += P.stt_s * sg[2] + P.stt_x * sz;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Sweep 1 (B5): n -> n^p.  Reads n (own + gathered neighbours), optional dipolar force of n; writes n^p and,
// with STORE_A, the rotation field A.
template <int BX, int BY, int BZ, bool STORE_A>
__global__ void __launch_bounds__(BX *BY *BZ)
    predictor_kernel(const __grid_constant__ DevicePlan P, const double *__restrict__ n, const double *__restrict__ fddi,
                     double *__restrict__ np, double *__restrict__ Aout, const unsigned long long *__restrict__ d_step,
                     unsigned int step_add) {
    const Site s = locate<BX, BY, BZ>(P);
    if (!s.valid) return;
    const int st = P.stride;
    const double *const cfg[1] = {n};
    const double own[1][3] = {{n[s.idx], n[st + s.idx], n[2 * st + s.idx]}};
    double F[1][3] = {{0.0, 0.0, 0.0}};
    short_range_force<1>(P, cfg, s, own, T_ALL, F);
    if (P.has_ddi) { F[0][0] += fddi[s.idx]; F[0][1] += fddi[st + s.idx]; F[0][2] += fddi[2 * st + s.idx]; }
    if (P.thermal_on) {
        double xi[3];
        thermal_xi(P.seed_lo, P.seed_hi, *d_step + step_add, (uint32_t)(s.b + P.nb * (s.idx - s.b * P.Ncell)), xi);
        const double sg = P.sigma[s.b];
        F[0][0] += sg * xi[0]; F[0][1] += sg * xi[1]; F[0][2] += sg * xi[2];
    }
    double sg[1][3] = {{0.0, 0.0, 0.0}};
    if (P.stt_on) stt_gradient<1>(P, cfg, s, own, sg);
    double A[3], out[3];
    rotation_field(P, s.b, own[0], F[0], sg[0], A);
    rodrigues(A, P.dt, P.dt2, own[0], out);
    np[s.idx] = out[0]; np[st + s.idx] = out[1]; np[2 * st + s.idx] = out[2];
    if (STORE_A) { Aout[s.idx] = A[0]; Aout[st + s.idx] = A[1]; Aout[2 * st + s.idx] = A[2]; }
}

// Sweep 2 (B6, B7): A^p = A(n^p) with the same thermal field, A^c = (A + A^p)/2, n(t+dt) = R(A^c) n(t), renormalise.
// Without STORE_A the predictor-stage A is recomputed from n (120 B per spin-update instead of 168 B).
template <int BX, int BY, int BZ, bool STORE_A>
__global__ void __launch_bounds__(BX *BY *BZ)
    corrector_kernel(const __grid_constant__ DevicePlan P, const double *__restrict__ n, const double *__restrict__ np,
                     const double *__restrict__ fddi_n, const double *__restrict__ fddi_np, const double *__restrict__ Ain,
                     double *__restrict__ nout, const unsigned long long *__restrict__ d_step, unsigned int step_add) {
    const Site s = locate<BX, BY, BZ>(P);
    if (!s.valid) return;
    const int st = P.stride;
    double xi[3] = {0.0, 0.0, 0.0};
    if (P.thermal_on) {
        thermal_xi(P.seed_lo, P.seed_hi, *d_step + step_add, (uint32_t)(s.b + P.nb * (s.idx - s.b * P.Ncell)), xi);
        const double sg = P.sigma[s.b];
        xi[0] *= sg; xi[1] *= sg; xi[2] *= sg;
    }
    double A[3], Ap[3];
    const double n0[3] = {n[s.idx], n[st + s.idx], n[2 * st + s.idx]};
    if (STORE_A) {
        const double *const cfg[1] = {np};
        const double own[1][3] = {{np[s.idx], np[st + s.idx], np[2 * st + s.idx]}};
        double F[1][3] = {{xi[0], xi[1], xi[2]}};
        short_range_force<1>(P, cfg, s, own, T_ALL, F);
        if (P.has_ddi) { F[0][0] += fddi_np[s.idx]; F[0][1] += fddi_np[st + s.idx]; F[0][2] += fddi_np[2 * st + s.idx]; }
        double sg[1][3] = {{0.0, 0.0, 0.0}};
        if (P.stt_on) stt_gradient<1>(P, cfg, s, own, sg);
        rotation_field(P, s.b, own[0], F[0], sg[0], Ap);
        A[0] = Ain[s.idx]; A[1] = Ain[st + s.idx]; A[2] = Ain[2 * st + s.idx];
    } else {
        const double *const cfg[2] = {n, np};
        const double own[2][3] = {{n0[0], n0[1], n0[2]}, {np[s.idx], np[st + s.idx], np[2 * st + s.idx]}};
        double F[2][3] = {{xi[0], xi[1], xi[2]}, {xi[0], xi[1], xi[2]}};
        short_range_force<2>(P, cfg, s, own, T_ALL, F);
        if (P.has_ddi) {
            F[0][0] += fddi_n[s.idx]; F[0][1] += fddi_n[st + s.idx]; F[0][2] += fddi_n[2 * st + s.idx];
            F[1][0] += fddi_np[s.idx]; F[1][1] += fddi_np[st + s.idx]; F[1][2] += fddi_np[2 * st + s.idx];
        }
        double sg[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
        if (P.stt_on) stt_gradient<2>(P, cfg, s, own, sg);
        rotation_field(P, s.b, own[0], F[0], sg[0], A);
        rotation_field(P, s.b, own[1], F[1], sg[1], Ap);
    }
    const double Ac[3] = {0.5 * (A[0] + Ap[0]), 0.5 * (A[1] + Ap[1]), 0.5 * (A[2] + Ap[2])};
    double out[3];
    rodrigues(Ac, P.dt, P.dt2, n0, out);
    renormalise(out);
    nout[s.idx] = out[0]; nout[st + s.idx] = out[1]; nout[2 * st + s.idx] = out[2];
}

// ---------------------------------------------------------------------------------------------------------
// Boundary order (AoS, basis fastest) <-> internal order (SoA, sublattice-major)
__global__ void pack_kernel(const double *__restrict__ aos, double *__restrict__ soa, int N, int nb, int Ncell, int stride, int normalise, int *bad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // boundary index
    if (i >= N) return;
    double v[3] = {aos[3 * (size_t)i], aos[3 * (size_t)i + 1], aos[3 * (size_t)i + 2]};
    if (normalise) {
        const double r2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
        if (!(r2 > 0.0) || !isfinite(r2)) { atomicExch(bad, 1); v[0] = 0; v[1] = 0; v[2] = 1; }
        else { const double r = sqrt(r2); v[0] /= r; v[1] /= r; v[2] /= r; }
    }
    const int b = i % nb, cell = i / nb, j = b * Ncell + cell;
    soa[j] = v[0]; soa[stride + j] = v[1]; soa[2 * stride + j] = v[2];
}
__global__ void unpack_kernel(const double *__restrict__ soa, double *__restrict__ aos, int N, int nb, int Ncell, int stride,
                              const double *__restrict__ scale /*per sublattice or null*/) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int b = i % nb, cell = i / nb, j = b * Ncell + cell;
    const double sc = scale ? scale[b] : 1.0;
    aos[3 * (size_t)i] = sc * soa[j]; aos[3 * (size_t)i + 1] = sc * soa[stride + j]; aos[3 * (size_t)i + 2] = sc * soa[2 * stride + j];
}

// deterministic force F (meV, SoA) of the current configuration: all terms of the mask (+ dipolar array if given)
template <int BX, int BY, int BZ>
__global__ void __launch_bounds__(BX *BY *BZ)
    force_kernel(const __grid_constant__ DevicePlan P, const double *__restrict__ n, const double *__restrict__ fddi, int mask,
                 double *__restrict__ Fout) {
    const Site s = locate<BX, BY, BZ>(P);
    if (!s.valid) return;
    const int st = P.stride;
    const double *const cfg[1] = {n};
    const double own[1][3] = {{n[s.idx], n[st + s.idx], n[2 * st + s.idx]}};
    double F[1][3] = {{0.0, 0.0, 0.0}};
    short_range_force<1>(P, cfg, s, own, mask, F);
    if ((mask & T_DDI) && P.has_ddi) { F[0][0] += fddi[s.idx]; F[0][1] += fddi[st + s.idx]; F[0][2] += fddi[2 * st + s.idx]; }
    Fout[s.idx] = F[0][0]; Fout[st + s.idx] = F[0][1]; Fout[2 * st + s.idx] = F[0][2];
}

// ---------------------------------------------------------------------------------------------------------
// Reductions: energies per term through Euler's identity E_k = -(1/k) sum_i n_i . F_i^(k) (k = 1 Zeeman, 2 anisotropy /
// exchange / DMI / dipolar, 4 quadruplets), magnetisation sum, max torque.  Warp shuffle, then one value per warp in shared
// memory, then one partial per block; a second single-block kernel folds the partials in a fixed order (deterministic).
constexpr int N_RED = 10;   // 6 energies, 3 magnetisation components, max torque

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

template <int BX, int BY, int BZ>
__global__ void __launch_bounds__(BX *BY *BZ)
    reduce_kernel(const __grid_constant__ DevicePlan P, const double *__restrict__ n, const double *__restrict__ fddi,
                  double *__restrict__ partials) {
    constexpr int NT = BX * BY * BZ, NW = NT / 32;
    __shared__ double sh[N_RED][NW];
    const Site s = locate<BX, BY, BZ>(P);
    double v[N_RED];
#pragma unroll
    for (int k = 0; k < N_RED; ++k) v[k] = 0.0;
    if (s.valid) {
        const int st = P.stride;
        const double *const cfg[1] = {n};
        const double own[1][3] = {{n[s.idx], n[st + s.idx], n[2 * st + s.idx]}};
        double Ft[3] = {0.0, 0.0, 0.0};
        const int masks[5] = {T_ZEE, T_ANI, T_EXC, T_DMI, T_QUAD};
        const double inv_k[5] = {1.0, 0.5, 0.5, 0.5, 0.25};
#pragma unroll
        for (int t = 0; t < 5; ++t) {
            double F[1][3] = {{0.0, 0.0, 0.0}};
            short_range_force<1>(P, cfg, s, own, masks[t], F);
            v[t] = -inv_k[t] * (own[0][0] * F[0][0] + own[0][1] * F[0][1] + own[0][2] * F[0][2]);
            Ft[0] += F[0][0]; Ft[1] += F[0][1]; Ft[2] += F[0][2];
        }
        if (P.has_ddi) {
            const double fx = fddi[s.idx], fy = fddi[st + s.idx], fz = fddi[2 * st + s.idx];
            v[5] = -0.5 * (own[0][0] * fx + own[0][1] * fy + own[0][2] * fz);
            Ft[0] += fx; Ft[1] += fy; Ft[2] += fz;
        }
        v[6] = own[0][0]; v[7] = own[0][1]; v[8] = own[0][2];
        const double p = Ft[0] * own[0][0] + Ft[1] * own[0][1] + Ft[2] * own[0][2];
        const double tx = Ft[0] - p * own[0][0], ty = Ft[1] - p * own[0][1], tz = Ft[2] - p * own[0][2];
        v[9] = sqrt(tx * tx + ty * ty + tz * tz);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < N_RED; ++k) {
        const double r = (k == 9) ? warp_max(v[k]) : warp_sum(v[k]);
        if (lane == 0) sh[k][w] = r;
    }
    __syncthreads();
    if (threadIdx.x < N_RED) {
        const int k = threadIdx.x;
        double r = sh[k][0];
        for (int i = 1; i < NW; ++i) r = (k == 9) ? fmax(r, sh[k][i]) : r + sh[k][i];
        partials[(size_t)(blockIdx.y * gridDim.x + blockIdx.x) * N_RED + k] = r;
    }
}

__global__ void reduce_final_kernel(const double *__restrict__ partials, int nblocks, double *__restrict__ out) {
    // one block of 32*N_RED threads: warp k folds column k in a fixed order
    const int k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (k >= N_RED) return;
    double r = 0.0;
    for (int i = lane; i < nblocks; i += 32) {
        const double x = partials[(size_t)i * N_RED + k];
        r = (k == 9) ? fmax(r, x) : r + x;
    }
    r = (k == 9) ? warp_max(r) : warp_sum(r);
    if (lane == 0) out[k] = r;
}

__global__ void advance_step_kernel(unsigned long long *d_step, unsigned long long add) { *d_step += add; }

}  // namespace spin
