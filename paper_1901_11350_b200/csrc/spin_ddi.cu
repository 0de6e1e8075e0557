// spin_ddi.cu -- dipole-dipole force by zero-padded FFT convolution.
//
// cuFFT performs only the transforms; the dipole-tensor build (image sums), the padding scatter, the 3x3 tensor x
// spin contraction in k-space and the field gather are hand-written kernels.
//
//   padded size   P_d = 2 N_d if N_d > 1 else 1                                     (R17)
//   tensor        K_ab(Delta) = sum_{images t} T(r),  r = alat ((Delta + t N) + p_a - p_b) . bravais,
//                 T(r) = (3 r^ r^T - 1)/r^3, Delta = target cell - source cell in (-N_d, N_d), stored at
//                 Delta mod P_d, index N_d left zero; r = 0 skipped                  (R16, R18)
//   force         F_a(c) = mu_a C_dd IFFT[ sum_b K^_ab(k) . FFT[mu_b n_b zero padded](k) ](c),  c in [0, N)
// One padded array per sublattice and one spectrum product per sublattice pair (:87).
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "spinllg_internal.h"

using namespace spin;

struct DdiState {
    int P[3];
    int64_t Ptot, Phalf;       // real points, complex points of the half spectrum
    int rank;                  // number of non-unit padded dimensions
    int fdims[3];              // cuFFT dims, slowest first
    cufftHandle plan_r2c, plan_c2r;
    bool have_plans;
    double *d_Mpad;            // [nb*3][Ptot]   real, zero outside the occupied corner
    double *d_Hpad;            // [nb*3][Ptot]   real result of the inverse transform
    cufftDoubleComplex *d_Mhat, *d_Hhat;   // [nb*3][Phalf]
    cufftDoubleComplex *d_Khat;            // [nb*nb][6][Phalf]
    double *d_geom;            // small device copy: bravais*alat (9), basis (3*nb), mu (nb)
    // ---- slab path (thin films, one basis atom): cuFFT transforms the a-b planes only (2-D, batched over the occupied
    // c-planes); the short transform along c, the tensor contraction and the inverse transform along c are one kernel.
    bool slab;
    int NZ, PZ;                // occupied planes, padded length along c (PZ = 2 NZ, or 1)
    int64_t S2, R2;            // complex / real points of one a-b plane: P1*(P0/2+1), P1*P0
    int SL, S1, S1p;           // slabs = 3 NZ (component x occupied plane); complex points of one row: P0/2+1; row pitch (128-byte multiple)
    // Layout of the slab path: [row ib][slab][ia or ka].  The a-pass (D2Z / Z2D, length P0) is batched over the Nb occupied rows
    // only (rows of zero padding are never transformed); the b-pass (Z2Z, length P1) runs over columns with stride SL*S1, batched
    // over (slab, ka).  Buffers: s_in real [Nb][SL][P0] (ia >= Na stays zero), s_a complex [P1][SL][S1p] (rows >= Nb stay zero),
    // s_b complex (b-pass output, contracted in place), s_d complex (inverse b-pass), s_out real [Nb][SL][P0].
    cufftHandle plan_a_fwd, plan_a_inv, plan_b;
    double *s_in, *s_out;
    cufftDoubleComplex *s_a, *s_b, *s_c, *s_d;
    double *d_Kre;             // [6][PZ][S2] real: the tensor spectrum is real for a single basis atom (the kernel is even)
    bool own_a;                // the a-pass is ddi_apass_fwd / ddi_apass_inv (rows of power-of-two length) instead of scatter + cuFFT + gather
    int a_rows_per_block;      // rows (warps) per block of those kernels
    size_t a_smem;
    double2 *d_tw;             // exp(-2 pi i t / P0), t < P0
    // fused b-pass (ddi_bfused_kernel): the a-pass kernels work in the transposed layout, s_a = [ka][slab][ib], s_d = the two partial
    // results [r][ka][slab][ib]; the full spectra and cuFFT's b-pass are not used
    bool fused_b;
    double2 *d_tw_b;           // exp(-2 pi i t / P1), t < P1
    double *d_Kb;              // [ka][r][6][planes][k'], ddi_bfused_tensor_kernel
    size_t bf_smem;
    bool a256, b256;           // rows / columns of length 256: the radix-16 kernels (ddi_apass256_*, ddi_bfused_kernel<.., true>)
    bool mirror;               // K(kz) = +-K(PZ - kz) (c perpendicular to the film): the contraction reads PZ/2 + 1 of the PZ planes
};

namespace {

template <int V> struct spin_ddi_int { static constexpr int value = V; };

struct DdiGeom {
    double brav[9];                      // rows, Angstrom
    double basis[3 * SPIN_MAX_BASIS];    // fractional
    int N[3], P[3], img[3];
};

// K_ab(Delta) summed over periodic images; one thread per padded grid point; 6 components written at stride Ptot.
__global__ void ddi_tensor_kernel(const __grid_constant__ DdiGeom G, int a, int b, long long Ptot, double *__restrict__ out) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= Ptot) return;
    const int g[3] = {(int)(idx % G.P[0]), (int)((idx / G.P[0]) % G.P[1]), (int)(idx / ((long long)G.P[0] * G.P[1]))};
    double acc[6] = {0, 0, 0, 0, 0, 0};
    bool skip = false;
    int Delta[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if (G.P[d] == 1) { Delta[d] = 0; continue; }
        if (g[d] == G.N[d]) skip = true;
        Delta[d] = (g[d] < G.N[d]) ? g[d] : g[d] - G.P[d];
    }
    if (!skip) {
        const double f0 = Delta[0] + G.basis[3 * a + 0] - G.basis[3 * b + 0];
        const double f1 = Delta[1] + G.basis[3 * a + 1] - G.basis[3 * b + 1];
        const double f2 = Delta[2] + G.basis[3 * a + 2] - G.basis[3 * b + 2];
        for (int t2 = -G.img[2]; t2 <= G.img[2]; ++t2)
            for (int t1 = -G.img[1]; t1 <= G.img[1]; ++t1)
                for (int t0 = -G.img[0]; t0 <= G.img[0]; ++t0) {
                    const double u0 = f0 + (double)t0 * G.N[0], u1 = f1 + (double)t1 * G.N[1], u2 = f2 + (double)t2 * G.N[2];
                    const double rx = u0 * G.brav[0] + u1 * G.brav[3] + u2 * G.brav[6];
                    const double ry = u0 * G.brav[1] + u1 * G.brav[4] + u2 * G.brav[7];
                    const double rz = u0 * G.brav[2] + u1 * G.brav[5] + u2 * G.brav[8];
                    const double r2 = rx * rx + ry * ry + rz * rz;
                    if (r2 < 1e-20) continue;
                    const double inv_r2 = 1.0 / r2, inv_r3 = inv_r2 / sqrt(r2), w = 3.0 * inv_r2 * inv_r3;
                    acc[0] += w * rx * rx - inv_r3; acc[1] += w * rx * ry; acc[2] += w * rx * rz;
                    acc[3] += w * ry * ry - inv_r3; acc[4] += w * ry * rz; acc[5] += w * rz * rz - inv_r3;
                }
    }
#pragma unroll
    for (int m = 0; m < 6; ++m) out[(size_t)m * Ptot + idx] = acc[m];
}

// M_b padded <- mu_b n_b on the occupied corner (the rest of the array stays zero from allocation time)
// (Ptot = stride between components: the whole padded grid, or NZ a-b planes on the slab path)
__global__ void ddi_scatter_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ n, int P0, int P1, long long Ptot,
                                   const double *__restrict__ mu, double *__restrict__ Mpad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // b*Ncell + cell, x fastest
    if (i >= L.nb * L.Ncell) return;
    const int b = i / L.Ncell, cell = i - b * L.Ncell;
    const int ia = cell % L.Na, ib = (cell / L.Na) % L.Nb, ic = cell / (L.Na * L.Nb);
    const long long p = ia + (long long)P0 * (ib + (long long)P1 * ic);
    const int j = b * L.sub + ((ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + (ia + L.LA);
    const double m = mu[b] * (L.mu_ratio ? L.mu_ratio[b + L.nb * cell] : 1.0);      // per-site moments
#pragma unroll
    for (int k = 0; k < 3; ++k) Mpad[(size_t)(b * 3 + k) * Ptot + p] = m * n[j + k * L.PA];
}

// H^_a = sum_b K^_ab . M^_b  (symmetric 3x3 complex tensor from 6 stored components)
__global__ void ddi_contract_kernel(const cufftDoubleComplex *__restrict__ Khat, const cufftDoubleComplex *__restrict__ Mhat,
                                    cufftDoubleComplex *__restrict__ Hhat, int nb, long long Phalf) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Phalf) return;
    const int a = blockIdx.y;
    double hr[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (int b = 0; b < nb; ++b) {
        const cufftDoubleComplex *K = Khat + (size_t)(a * nb + b) * 6 * Phalf;
        const cufftDoubleComplex m0 = Mhat[(size_t)(b * 3 + 0) * Phalf + q], m1 = Mhat[(size_t)(b * 3 + 1) * Phalf + q],
                                 m2 = Mhat[(size_t)(b * 3 + 2) * Phalf + q];
        const cufftDoubleComplex kxx = K[q], kxy = K[Phalf + q], kxz = K[2 * Phalf + q], kyy = K[3 * Phalf + q],
                                 kyz = K[4 * Phalf + q], kzz = K[5 * Phalf + q];
        hr[0] += kxx.x * m0.x - kxx.y * m0.y + kxy.x * m1.x - kxy.y * m1.y + kxz.x * m2.x - kxz.y * m2.y;
        hi[0] += kxx.x * m0.y + kxx.y * m0.x + kxy.x * m1.y + kxy.y * m1.x + kxz.x * m2.y + kxz.y * m2.x;
        hr[1] += kxy.x * m0.x - kxy.y * m0.y + kyy.x * m1.x - kyy.y * m1.y + kyz.x * m2.x - kyz.y * m2.y;
        hi[1] += kxy.x * m0.y + kxy.y * m0.x + kyy.x * m1.y + kyy.y * m1.x + kyz.x * m2.y + kyz.y * m2.x;
        hr[2] += kxz.x * m0.x - kxz.y * m0.y + kyz.x * m1.x - kyz.y * m1.y + kzz.x * m2.x - kzz.y * m2.y;
        hi[2] += kxz.x * m0.y + kxz.y * m0.x + kyz.x * m1.y + kyz.y * m1.x + kzz.x * m2.y + kzz.y * m2.x;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) Hhat[(size_t)(a * 3 + k) * Phalf + q] = make_cuDoubleComplex(hr[k], hi[k]);
}

// F_a(c) = mu_a C_dd / Ptot * H_a(c) on the occupied corner, written in the internal SoA layout
__global__ void ddi_gather_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ Hpad, int P0, int P1, long long Ptot,
                                  const double *__restrict__ mu, double scale, double *__restrict__ f) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= L.nb * L.Ncell) return;
    const int b = i / L.Ncell, cell = i - b * L.Ncell;
    const int ia = cell % L.Na, ib = (cell / L.Na) % L.Nb, ic = cell / (L.Na * L.Nb);
    const long long p = ia + (long long)P0 * (ib + (long long)P1 * ic);
    const int j = b * L.sub + ((ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + (ia + L.LA);
    const double m = mu[b] * scale * (L.mu_ratio ? L.mu_ratio[b + L.nb * cell] : 1.0);
#pragma unroll
    for (int k = 0; k < 3; ++k) f[j + k * L.PA] = m * Hpad[(size_t)(b * 3 + k) * Ptot + p];
}

// slab path: the same two copies in the row-interleaved layout [ib][slab = (b 3 + comp) NZ + ic][ia]
__global__ void ddi_slab_scatter_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ n, int P0, int SL, const double *__restrict__ mu,
                                        double *__restrict__ in) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;      // b * Ncell + cell
    if (i >= L.nb * L.Ncell) return;
    const int b = i / L.Ncell, cell = i - b * L.Ncell;
    const int ia = cell % L.Na, ib = (cell / L.Na) % L.Nb, ic = cell / (L.Na * L.Nb);
    const int j = b * L.sub + ((ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + (ia + L.LA);
    const double m = mu[b] * (L.mu_ratio ? L.mu_ratio[b + L.nb * cell] : 1.0);
#pragma unroll
    for (int k = 0; k < 3; ++k) in[((size_t)ib * SL + ((b * 3 + k) * L.Nc + ic)) * P0 + ia] = m * n[j + k * L.PA];
}
__global__ void ddi_slab_gather_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ out, int P0, int SL, const double *__restrict__ mu,
                                       double scale, double *__restrict__ f) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= L.nb * L.Ncell) return;
    const int b = i / L.Ncell, cell = i - b * L.Ncell;
    const int ia = cell % L.Na, ib = (cell / L.Na) % L.Nb, ic = cell / (L.Na * L.Nb);
    const int j = b * L.sub + ((ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + (ia + L.LA);
    const double m = mu[b] * scale * (L.mu_ratio ? L.mu_ratio[b + L.nb * cell] : 1.0);
#pragma unroll
    for (int k = 0; k < 3; ++k) f[j + k * L.PA] = m * out[((size_t)ib * SL + ((b * 3 + k) * L.Nc + ic)) * P0 + ia];
}


// ---------------------------------------------------------------------------------------------------------------------------
// The a-pass of the slab path, hand-written for power-of-two rows ("FFTs ... power of two"): the padding scatter and the
// transform along a are one kernel, the inverse transform and the field gather another.  A row holds Na real values followed by Na zeros
// (P0 = 2 Na); its transform is taken as ONE complex transform of length M = P0 / 2 = Na of z(j) = x(2j) + i x(2j+1) (only j < M / 2 is
// non-zero) followed by the usual split  X(k) = E(k) + W^k O(k),  E = (Z(k) + Z*(M-k)) / 2,  O = (Z(k) - Z*(M-k)) / (2i),  W = exp(-2 pi i / P0).
// One warp per row; the complex transform is a Stockham autosort (radix 8, closed by one pass of radix 4 or 2) ping-ponging between two
// padded shared-memory rows, the first twiddle of a butterfly from a table of exp(-2 pi i t / P0) in global memory.  Compared with scatter + cuFFT D2Z this reads the
// spins once where they live (no padded real copy: 12.6 instead of 12.6 + 12.6 + 25.2 MB on cfg5) and launches one kernel instead of two.
// Programmatic dependent launch (fused path): the kernels of an evaluation are launched with programmatic stream serialisation, so the
// blocks of the next kernel become resident while the previous one drains and run their prologue (tables, tensor prefetch); everything
// that reads the previous kernel's output comes after this wait (a no-op in a kernel launched the plain way).
__device__ __forceinline__ void ddi_wait_upstream() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ double2 ddi_cadd(const double2 a, const double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 ddi_csub(const double2 a, const double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 ddi_cmul(const double2 a, const double2 b) { return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x)); }
// times -i (forward, SIGN < 0) or +i (inverse)
template <int SIGN> __device__ __forceinline__ double2 ddi_rot90(const double2 a) { return SIGN < 0 ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x); }
// times exp(SIGN i pi / 4)
template <int SIGN> __device__ __forceinline__ double2 ddi_rot45(const double2 a) {
    const double h = 0.70710678118654752440;
    return SIGN < 0 ? make_double2(h * (a.x + a.y), h * (a.y - a.x)) : make_double2(h * (a.x - a.y), h * (a.y + a.x));
}
// shared-memory rows are padded by one element in eight: the stores of the first passes (stride R elements between lanes) and the loads
// (consecutive elements) are then both free of bank conflicts for 16-byte elements
__device__ __forceinline__ int ddi_pad(const int i) { return i + (i >> 3); }

// One butterfly of radix R (8, 4 or 2): v[r] times w1^r (twiddle = false: w1 = 1), then the R-point transform.  Result r of the transform
// is left in v[ddi_perm<R>(r)]... read it through ddi_out<R>(r): the position in v that holds output r.
template <int R> __host__ __device__ constexpr int ddi_out(int r) { return R == 8 ? ((r & 1) << 2 | (r & 2) | (r & 4) >> 2) : (R == 4 ? ((r & 1) << 1 | (r & 2) >> 1) : r); }
template <int SIGN, int R>      // SIGN -1 forward, +1 inverse (unnormalised)
__device__ __forceinline__ void ddi_butterfly(double2 (&v)[R], const bool twiddle, const double2 w1) {
    if constexpr (R == 8) {
        if (twiddle) {
            const double2 w2 = ddi_cmul(w1, w1), w3 = ddi_cmul(w2, w1), w4 = ddi_cmul(w2, w2);
            v[1] = ddi_cmul(v[1], w1); v[2] = ddi_cmul(v[2], w2); v[3] = ddi_cmul(v[3], w3); v[4] = ddi_cmul(v[4], w4);
            v[5] = ddi_cmul(v[5], ddi_cmul(w4, w1)); v[6] = ddi_cmul(v[6], ddi_cmul(w3, w3)); v[7] = ddi_cmul(v[7], ddi_cmul(w4, w3));
        }
        // three radix-2 stages, result in bit-reversed order
        double2 t;
        t = ddi_csub(v[0], v[4]); v[0] = ddi_cadd(v[0], v[4]); v[4] = t;
        t = ddi_csub(v[1], v[5]); v[1] = ddi_cadd(v[1], v[5]); v[5] = ddi_rot45<SIGN>(t);
        t = ddi_csub(v[2], v[6]); v[2] = ddi_cadd(v[2], v[6]); v[6] = ddi_rot90<SIGN>(t);
        t = ddi_csub(v[3], v[7]); v[3] = ddi_cadd(v[3], v[7]); v[7] = ddi_rot90<SIGN>(ddi_rot45<SIGN>(t));
#pragma unroll
        for (int h = 0; h < 8; h += 4) {
            t = ddi_csub(v[h], v[h + 2]); v[h] = ddi_cadd(v[h], v[h + 2]); v[h + 2] = t;
            t = ddi_csub(v[h + 1], v[h + 3]); v[h + 1] = ddi_cadd(v[h + 1], v[h + 3]); v[h + 3] = ddi_rot90<SIGN>(t);
        }
#pragma unroll
        for (int h = 0; h < 8; h += 2) { t = ddi_csub(v[h], v[h + 1]); v[h] = ddi_cadd(v[h], v[h + 1]); v[h + 1] = t; }
    } else if constexpr (R == 4) {
        if (twiddle) { const double2 w2 = ddi_cmul(w1, w1); v[1] = ddi_cmul(v[1], w1); v[2] = ddi_cmul(v[2], w2); v[3] = ddi_cmul(v[3], ddi_cmul(w2, w1)); }
        const double2 t0 = ddi_cadd(v[0], v[2]), t1 = ddi_csub(v[0], v[2]), t2 = ddi_cadd(v[1], v[3]), t3 = ddi_rot90<SIGN>(ddi_csub(v[1], v[3]));
        v[0] = ddi_cadd(t0, t2); v[2] = ddi_cadd(t1, t3); v[1] = ddi_csub(t0, t2); v[3] = ddi_csub(t1, t3);      // bit-reversed: v[2] holds output 1
    } else {
        if (twiddle) v[1] = ddi_cmul(v[1], w1);
        const double2 t = ddi_csub(v[0], v[1]);
        v[0] = ddi_cadd(v[0], v[1]); v[1] = t;
    }
}

// One Stockham pass of radix R of a transform of length M = 2^lgM by one warp: element i of the source is ld(i), element i of the
// destination goes to st(i, v) (natural index; shared-memory rows, or global memory for the first / last pass of a fused kernel).
// Ns = 2^lgNs = product of the radices of the passes before this one.  Twiddles exp(SIGN 2 pi i k r / (Ns R)): the first power from the
// table tw[t] = exp(-2 pi i t / (2 M)), the others by multiplication (depth 3).  Index arithmetic is shifts and masks only.
// INPLACE: source and destination are the same row -- every lane loads all its butterflies (at most NB, i.e. M <= 32 NB R; the fused kernel: M <= 256), the warp
// synchronises, then the lanes store; otherwise butterfly by butterfly (NB is ignored).
template <int SIGN, int R, class Store>
__device__ __forceinline__ void ddi_fft_finish(double2 (&v)[R], const int j, const int lgNs, const int tshift, const double2 *__restrict__ tw, Store &&st) {
    constexpr int lgR = R == 8 ? 3 : (R == 4 ? 2 : 1);
    const int k = j & ((1 << lgNs) - 1), j0 = ((j - k) << lgR) + k;
    double2 w1 = make_double2(1.0, 0.0);
    if (k) { w1 = tw[k << tshift]; if (SIGN > 0) w1.y = -w1.y; }
    ddi_butterfly<SIGN, R>(v, k != 0, w1);
#pragma unroll
    for (int r = 0; r < R; ++r) st(j0 + (r << lgNs), v[ddi_out<R>(r)]);
}
template <int SIGN, int R, bool INPLACE, int NB, class Load, class Store>
__device__ __forceinline__ void ddi_fft_pass(const int lgM, const int lgNs, const double2 *__restrict__ tw, const int lane, Load &&ld, Store &&st) {
    constexpr int lgR = R == 8 ? 3 : (R == 4 ? 2 : 1);
    const int span = 1 << (lgM - lgR), tshift = lgM - lgNs - lgR + 1;
    if constexpr (INPLACE) {
        double2 v[NB][R];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int j = min(lane + 32 * b, span - 1);      // idle lanes load a valid element too (a guarded load costs ptxas 1.5 KB of spills)
#pragma unroll
            for (int r = 0; r < R; ++r) v[b][r] = ld(j + (r << (lgM - lgR)));
        }
        __syncwarp();
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int j = lane + 32 * b;
            if (j < span) ddi_fft_finish<SIGN, R>(v[b], j, lgNs, tshift, tw, st);
        }
    } else {
        for (int j = lane; j < span; j += 32) {
            double2 v[R];
#pragma unroll
            for (int r = 0; r < R; ++r) v[r] = ld(j + (r << (lgM - lgR)));
            ddi_fft_finish<SIGN, R>(v, j, lgNs, tshift, tw, st);
        }
    }
}
// radix of the pass that follows passes of product 2^lgNs: 8 while it divides what is left, then 4 or 2
__host__ __device__ __forceinline__ int ddi_radix(const int lgM, const int lgNs) { const int rem = lgM - lgNs; return rem >= 3 ? 8 : (rem == 2 ? 4 : 2); }
// the pass after passes of product 2^lgNs, whatever its radix; returns log2 of that radix
template <int SIGN, bool INPLACE, class Load, class Store>
__device__ __forceinline__ int ddi_fft_next_pass(const int lgM, const int lgNs, const double2 *__restrict__ tw, const int lane, Load &&ld, Store &&st) {
    const int R = ddi_radix(lgM, lgNs);
    if (R == 8) { ddi_fft_pass<SIGN, 8, INPLACE, 1>(lgM, lgNs, tw, lane, ld, st); return 3; }      // in place: M <= 256 = 32 lanes x 8 elements
    if (R == 4) { ddi_fft_pass<SIGN, 4, INPLACE, 2>(lgM, lgNs, tw, lane, ld, st); return 2; }
    ddi_fft_pass<SIGN, 2, INPLACE, 4>(lgM, lgNs, tw, lane, ld, st);
    return 1;
}

// One warp, complex transform of length M = 2^lgM >= 8 as a Stockham autosort, ping-ponging between the padded shared-memory rows
// a and b; returns the row that holds the result (natural order).
template <int SIGN>
__device__ __forceinline__ double2 *ddi_warp_fft(double2 *a, double2 *b, const int lgM, const double2 *__restrict__ tw, const int lane) {
    for (int lgNs = 0; lgNs < lgM;) {
        lgNs += ddi_fft_next_pass<SIGN, false>(lgM, lgNs, tw, lane, [&](int i) { return a[ddi_pad(i)]; }, [&](int i, const double2 v) { b[ddi_pad(i)] = v; });
        __syncwarp();
        double2 *t = a; a = b; b = t;
    }
    return a;
}

// per-site moment ratios of the sites 2j, 2j+1 of row (b, ib, ic) in boundary order b + nb * cell (one vector load for one sublattice)
__device__ __forceinline__ double2 ddi_row_ratio(const DevicePlan &L, int b, int ib, int ic, int j) {
    const size_t cell0 = (size_t)L.Na * (ib + (size_t)L.Nb * ic) + 2 * (size_t)j;
    if (L.nb == 1) return __ldg((const double2 *)(L.mu_ratio + cell0));
    return make_double2(__ldg(L.mu_ratio + b + (size_t)L.nb * cell0), __ldg(L.mu_ratio + b + (size_t)L.nb * (cell0 + 1)));
}

// rows = Nb * SL occupied rows, slab = (b 3 + comp) Nc + ic.
// TR = false: row = ib SL + slab, element k of the row at row * S1p + k, k = 0 .. M (the layout cuFFT's b-pass works on).
// TR = true (fused b-pass): a block takes rows_per_block consecutive ib of ONE slab and writes [ka][slab][ib] -- its warps' results go
// through shared memory so that consecutive lanes write consecutive ib (whole 32-byte sectors and more).  `nbr` = Nb.
template <bool TR>
__global__ void __launch_bounds__(256) ddi_apass_fwd_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ n, int M, int SL, int S1p, int rows,
                                                            int rows_per_block, const double *__restrict__ mu_b, const double2 *__restrict__ tw,
                                                            cufftDoubleComplex *__restrict__ out) {
    extern __shared__ double2 ddi_sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row = blockIdx.x * rows_per_block + warp;
    if (!TR && (warp >= rows_per_block || row >= rows)) return;      // (TR: rows is a multiple of rows_per_block, every warp has a row)
    const int ib = TR ? row % L.Nb : row / SL, slab = TR ? row / L.Nb : row - ib * SL;
    const int bc = slab / L.Nc, ic = slab - bc * L.Nc, sb = bc / 3, comp = bc - 3 * sb;
    const double mu = mu_b[sb];
    const double2 *src = (const double2 *)(n + (size_t)sb * L.sub + ((size_t)(ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + comp * L.PA + L.LA);
    const int MP = M + (M >> 3), WS = 2 * MP + 1;       // padded row; buffers of a warp (the odd stride keeps the transposed reads conflict-free)
    double2 *a = ddi_sm + (size_t)warp * WS, *b = a + MP;
    for (int j = M / 2 + lane; j < M; j += 32) a[ddi_pad(j)] = make_double2(0.0, 0.0);      // the zero padding of the row
    ddi_wait_upstream();
#pragma unroll 4
    for (int j = lane; j < M / 2; j += 32) {                                                  // (unrolled: the loads of a lane are in flight together)
        double2 v = __ldg(src + j);
        double m0 = mu, m1 = mu;
        if (L.mu_ratio) { const double2 r = ddi_row_ratio(L, sb, ib, ic, j); m0 *= r.x; m1 *= r.y; }
        v.x *= m0; v.y *= m1;
        a[ddi_pad(j)] = v;
    }
    __syncwarp();
    const double2 *Z = ddi_warp_fft<-1>(a, b, 31 - __clz(M), tw, lane);
    double2 *X = (Z == a) ? b : a;                       // TR: the half spectrum of the row, unpadded, in the warp's other buffer
    cufftDoubleComplex *dst = out + (size_t)row * S1p;
    for (int k = lane; k <= M; k += 32) {
        const double2 zk = Z[ddi_pad(k & (M - 1))], zm = Z[ddi_pad((M - k) & (M - 1))];
        const double er = 0.5 * (zk.x + zm.x), ei = 0.5 * (zk.y - zm.y);            // E = (Z(k) + conj Z(M-k)) / 2
        const double orr = 0.5 * (zk.y + zm.y), oi = -0.5 * (zk.x - zm.x);          // O = (Z(k) - conj Z(M-k)) / (2i)
        const double2 w = __ldg(tw + k);                                            // exp(-2 pi i k / P0)
        const double2 x = make_double2(er + fma(orr, w.x, -oi * w.y), ei + fma(orr, w.y, oi * w.x));
        if (TR) X[k] = x; else dst[k] = x;
    }
    if (TR) {
        __syncthreads();
        const int xoff = (int)(X - a);                   // the same for every warp (same number of passes)
        const int ib0 = (blockIdx.x * rows_per_block) % L.Nb;
        const int lgr = __ffs(rows_per_block) - 1;       // (a power of two)
        cufftDoubleComplex *o = out + (size_t)slab * L.Nb + ib0;
        for (int idx = threadIdx.x; idx < (M + 1) << lgr; idx += blockDim.x) {
            const int k = idx >> lgr, w = idx & (rows_per_block - 1);
            o[(size_t)k * SL * L.Nb + w] = ddi_sm[w * WS + xoff + k];
        }
    }
}

// inverse: from the half spectrum X(k), k = 0 .. M, of every occupied row to P0 x(ia), ia < Na, scaled and written as the dipolar force.
// TR = true: the input is the two partial results of ddi_bfused_kernel, [r][ka][slab][ib] (in + part1 apart), added while loading.
template <bool TR>
__global__ void __launch_bounds__(256) ddi_apass_inv_kernel(const __grid_constant__ DevicePlan L, const cufftDoubleComplex *__restrict__ in, int M, int SL, int S1p,
                                                            int rows, int rows_per_block, const double *__restrict__ mu_b, double scale0, const double2 *__restrict__ tw,
                                                            double *__restrict__ f, size_t part1) {
    extern __shared__ double2 ddi_sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row = blockIdx.x * rows_per_block + warp;
    if (!TR && (warp >= rows_per_block || row >= rows)) return;
    const int ib = TR ? row % L.Nb : row / SL, slab = TR ? row / L.Nb : row - ib * SL;
    const int bc = slab / L.Nc, ic = slab - bc * L.Nc, sb = bc / 3, comp = bc - 3 * sb;
    const double scale = mu_b[sb] * scale0;
    const int MP = M + (M >> 3), WS = 2 * MP + 1;
    double2 *a = ddi_sm + (size_t)warp * WS, *b = a + MP;
    const cufftDoubleComplex *src = TR ? b : in + (size_t)row * S1p;                // TR: the row's half spectrum, gathered into b first
    ddi_wait_upstream();
    if (TR) {
        const int ib0 = (blockIdx.x * rows_per_block) % L.Nb;
        const int lgr = __ffs(rows_per_block) - 1, total = (M + 1) << lgr;      // (a power of two)
        const cufftDoubleComplex *g0 = in + (size_t)slab * L.Nb + ib0, *g1 = g0 + part1;
        constexpr int U = 4;                                 // loads of U elements in flight per thread
        for (int base = threadIdx.x; base < total; base += U * blockDim.x) {
            double2 p0[U], p1[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int idx = min(base + u * (int)blockDim.x, total - 1);
                const size_t o = (size_t)(idx >> lgr) * SL * L.Nb + (idx & (rows_per_block - 1));
                p0[u] = __ldg(g0 + o); p1[u] = __ldg(g1 + o);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int idx = base + u * (int)blockDim.x;
                if (idx < total) ddi_sm[(idx & (rows_per_block - 1)) * WS + MP + (idx >> lgr)] = make_double2(p0[u].x + p1[u].x, p0[u].y + p1[u].y);
            }
        }
        __syncthreads();
    }
    for (int k = lane; k < M; k += 32) {
        const cufftDoubleComplex xk = src[k], xm = src[M - k];
        const double er = xk.x + xm.x, ei = xk.y - xm.y;                            // E = X(k) + conj X(M-k)
        const double dr = xk.x - xm.x, di = xk.y + xm.y;                            // X(k) - conj X(M-k)
        const double2 w = __ldg(tw + k);                                            // times exp(+2 pi i k / P0)
        const double orr = fma(dr, w.x, di * w.y), oi = fma(di, w.x, -dr * w.y);
        a[ddi_pad(k)] = make_double2(er - oi, ei + orr);                            // Z = E + i O
    }
    __syncwarp();
    const double2 *z = ddi_warp_fft<+1>(a, b, 31 - __clz(M), tw, lane);
    double2 *dst = (double2 *)(f + (size_t)sb * L.sub + ((size_t)(ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + comp * L.PA + L.LA);
    for (int j = lane; j < M / 2; j += 32) {
        const double2 v = z[ddi_pad(j)];
        double m0 = scale, m1 = scale;
        if (L.mu_ratio) { const double2 r = ddi_row_ratio(L, sb, ib, ic, j); m0 *= r.x; m1 *= r.y; }
        dst[j] = make_double2(m0 * v.x, m1 * v.y);
    }
}

// rank-0 case (a single cell): the "transform" of one point is the point itself
__global__ void real_to_complex_kernel(const double *__restrict__ in, cufftDoubleComplex *__restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_cuDoubleComplex(in[i], 0.0);
}
__global__ void complex_to_real_kernel(const cufftDoubleComplex *__restrict__ in, double *__restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i].x;
}

// real part of a spectrum (slab path: the tensor spectrum of a single basis atom is real)
__global__ void real_part_kernel(const cufftDoubleComplex *__restrict__ in, double *__restrict__ out, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = in[i].x;
}

// twiddles exp(-2 pi i t / PZ), t < PZ, for every padded length along c the slab path takes (PZ <= 16), indexed [PZ][t].  The table is
// a function of PZ alone, so every system of the process shares it (films of different thickness may be alive at the same time).
__constant__ double DDI_TWR[17][16], DDI_TWI[17][16];

__host__ __device__ constexpr bool ddi_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
// (re + i im) times exp(-2 pi i a / 16).  Called with `a` known after unrolling, so the switch folds away: quarter turns cost nothing,
// eighth turns two additions and two products, the others a full complex product with literal constants.  The power-of-two lengths along c
// (PZ = 2, 4, 8, 16) take their twiddles from here instead of the table: of the 12 butterflies of a length-8 transform only 2 multiply.
__device__ __forceinline__ void ddi_rot16(const int a, double &re, double &im) {
    const double h = 0.70710678118654752440, c = 0.92387953251128675613, s = 0.38268343236508977173;      // cos pi/4, cos pi/8, sin pi/8
    const double r = re, i = im;
    double cw = 0.0, sw = 0.0;
    switch (a & 15) {
        case 0: return;
        case 4: re = i; im = -r; return;
        case 8: re = -r; im = -i; return;
        case 12: re = -i; im = r; return;
        case 2: re = h * (r + i); im = h * (i - r); return;
        case 6: re = h * (i - r); im = -h * (r + i); return;
        case 10: re = -h * (r + i); im = h * (r - i); return;
        case 14: re = h * (r - i); im = h * (r + i); return;
        case 1: cw = c; sw = s; break;
        case 3: cw = s; sw = c; break;
        case 5: cw = -s; sw = c; break;
        case 7: cw = -c; sw = s; break;
        case 9: cw = -c; sw = -s; break;
        case 11: cw = -s; sw = -c; break;
        case 13: cw = s; sw = -c; break;
        default: cw = c; sw = -s; break;
    }
    re = fma(r, cw, i * sw); im = fma(i, cw, -r * sw);
}
__host__ __device__ constexpr int ddi_bitrev(int p, int n) {      // n a power of two
    int r = 0;
    for (int b = 1, c = n >> 1; b < n; b <<= 1, c >>= 1) if (p & b) r |= c;
    return r;
}
// position of frequency j in the array the forward transform leaves (bit reversed for powers of two, natural otherwise; an involution)
template <int N> __host__ __device__ constexpr int ddi_pos(int j) { return ddi_pow2(N) ? ddi_bitrev(j, N) : j; }

// y(j) = sum_z x(z) W_N^(j z), W_N = exp(-2 pi i / N) = W_PZ^2 (PZ = 2 N), in place.  Powers of two: radix-2 decimation in frequency, the
// result is left in bit-reversed order; other lengths (3, 5, 6, 7): the plain sum, natural order.  Fully unrolled: x stays in registers.
template <int N>
__device__ __forceinline__ void ddi_dft_fwd(double (&re)[N], double (&im)[N]) {
    constexpr int PZ = 2 * N;
    if constexpr (ddi_pow2(N)) {
#pragma unroll
        for (int half = N / 2; half >= 1; half /= 2)
#pragma unroll
            for (int base = 0; base < N; base += 2 * half)
#pragma unroll
                for (int j = 0; j < half; ++j) {
                    const int t = j * (N / (2 * half)) * 2;      // W_(2 half)^j as a power of W_PZ
                    const double ar = re[base + j], ai = im[base + j], br = re[base + j + half], bi = im[base + j + half];
                    re[base + j] = ar + br; im[base + j] = ai + bi;
                    re[base + j + half] = ar - br; im[base + j + half] = ai - bi;
                    ddi_rot16(t * (16 / PZ), re[base + j + half], im[base + j + half]);
                }
    } else {
        double yr[N], yi[N];
#pragma unroll
        for (int j = 0; j < N; ++j) {
            double sr = 0.0, si = 0.0;
#pragma unroll
            for (int z = 0; z < N; ++z) {
                const int t = (2 * j * z) % PZ;
                const double wr = DDI_TWR[PZ][t], wi = DDI_TWI[PZ][t];
                sr = fma(re[z], wr, fma(-im[z], wi, sr)); si = fma(re[z], wi, fma(im[z], wr, si));
            }
            yr[j] = sr; yi[j] = si;
        }
#pragma unroll
        for (int j = 0; j < N; ++j) { re[j] = yr[j]; im[j] = yi[j]; }
    }
}
// x(z) = sum_j y(j) W_N^(-j z), unnormalised, from the order ddi_dft_fwd leaves to natural order, in place
template <int N>
__device__ __forceinline__ void ddi_dft_inv(double (&re)[N], double (&im)[N]) {
    constexpr int PZ = 2 * N;
    if constexpr (ddi_pow2(N)) {
#pragma unroll
        for (int half = 1; half < N; half *= 2)
#pragma unroll
            for (int base = 0; base < N; base += 2 * half)
#pragma unroll
                for (int j = 0; j < half; ++j) {
                    const int t = j * (N / (2 * half)) * 2;
                    double br = re[base + j + half], bi = im[base + j + half];
                    ddi_rot16(16 - t * (16 / PZ), br, bi);                         // conjugate twiddle
                    const double ar = re[base + j], ai = im[base + j];
                    re[base + j] = ar + br; im[base + j] = ai + bi;
                    re[base + j + half] = ar - br; im[base + j + half] = ai - bi;
                }
    } else {
        double yr[N], yi[N];
#pragma unroll
        for (int z = 0; z < N; ++z) {
            double sr = 0.0, si = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) {
                const int t = (2 * j * z) % PZ;
                const double wr = DDI_TWR[PZ][t], wi = -DDI_TWI[PZ][t];
                sr = fma(re[j], wr, fma(-im[j], wi, sr)); si = fma(re[j], wi, fma(im[j], wr, si));
            }
            yr[z] = sr; yi[z] = si;
        }
#pragma unroll
        for (int z = 0; z < N; ++z) { re[z] = yr[z]; im[z] = yi[z]; }
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// Transforms of length 256 (the a- and b-direction of a 256 x 256 film): two passes of radix 16 by HALF a warp, one butterfly of 16
// points per lane and pass, the row in place in shared memory.  x(n), n = l + 16 q;  X(p + 16 u) = sum_l [W^(l p) A(l, p)] W_16^(l u),
// A(l, p) = sum_q x(l + 16 q) W_16^(q p),  W = exp(-+ 2 pi i / 256).  Pass 1: lane l transforms its 16 inputs over q, multiplies by
// W^(l p) (table T[p - 1][l] in shared memory, conflict-free) and stores A(l, p) at l 16 + p; pass 2: lane p reads A(l, p) over l,
// transforms, and holds X(p + 16 u).  Rows are padded by one element in 16 (position i + (i >> 4)): every access of the 16 lanes is then
// either to consecutive elements or at a stride of 17 elements, both free of bank conflicts.  Against three passes of radix 8 / 8 / 4 by
// a whole warp this is two instead of three round trips through shared memory, one instead of two twiddle stages, and no index
// arithmetic beyond constant offsets.
__device__ __forceinline__ int ddi_pad16(const int i) { return i + (i >> 4); }
constexpr int DDI_LP256 = 272;             // 256 + 256 / 16
// in-place 4-point transform, natural order
template <int SIGN> __device__ __forceinline__ void ddi_dft4(double2 &a, double2 &b, double2 &c, double2 &d) {
    const double2 t0 = ddi_cadd(a, c), t1 = ddi_csub(a, c), t2 = ddi_cadd(b, d), t3 = ddi_rot90<SIGN>(ddi_csub(b, d));
    a = ddi_cadd(t0, t2); b = ddi_cadd(t1, t3); c = ddi_csub(t0, t2); d = ddi_csub(t1, t3);
}
// 16-point transform in registers: input v[n] in natural order, output k left in v[ddi_out16(k)].  HALF: v[8..15] are zero (not read).
__host__ __device__ constexpr int ddi_out16(int k) { return ((k & 3) << 2) | (k >> 2); }
template <int SIGN, bool HALF>
__device__ __forceinline__ void ddi_fft16(double2 (&v)[16]) {
    // over m for every s: (v[s], v[s+4], v[s+8], v[s+12]) -> A(s, t) in v[s + 4 t]
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        if constexpr (HALF) {
            const double2 a = v[s], b = v[s + 4], rb = ddi_rot90<SIGN>(b);
            v[s] = ddi_cadd(a, b); v[s + 4] = ddi_cadd(a, rb); v[s + 8] = ddi_csub(a, b); v[s + 12] = ddi_csub(a, rb);
        } else ddi_dft4<SIGN>(v[s], v[s + 4], v[s + 8], v[s + 12]);
    }
    // times W_16^(s t), then over s for every t: X(t + 4 u) in v[4 t + u]
#pragma unroll
    for (int t = 1; t < 4; ++t)
#pragma unroll
        for (int s = 1; s < 4; ++s) ddi_rot16(SIGN < 0 ? s * t : 16 - s * t, v[s + 4 * t].x, v[s + 4 * t].y);
    // the four values of one t sit at v[4 t' ...]: gather them as (v[0 + 4t], v[1 + 4t], v[2 + 4t], v[3 + 4t])
#pragma unroll
    for (int t = 0; t < 4; ++t) ddi_dft4<SIGN>(v[4 * t], v[4 * t + 1], v[4 * t + 2], v[4 * t + 3]);
}
// the table of pass 1: T[(p - 1) 16 + l] = exp(-2 pi i l p / 256) = tw[2 l p] of the table exp(-2 pi i t / 512); `nthreads` threads fill it
__device__ __forceinline__ void ddi_fill_t256(double2 *T, const double2 *__restrict__ tw, const int tid, const int nthreads) {
    for (int i = tid; i < 240; i += nthreads) T[i] = __ldg(tw + 2 * (i & 15) * ((i >> 4) + 1));
}
// pass 1 on the inputs v[q] = x(l + 16 q) of lane l: transform, twiddle, store A(l, p) into the row.  The caller has loaded v.
template <int SIGN, bool HALF>
__device__ __forceinline__ void ddi_fft256_pass1(double2 (&v)[16], double2 *row, const double2 *T, const int l) {
    ddi_fft16<SIGN, HALF>(v);
    double2 *dst = row + 17 * l;                  // ddi_pad16(16 l + p) = 17 l + p
    dst[0] = v[ddi_out16(0)];
#pragma unroll
    for (int p = 1; p < 16; ++p) {
        double2 w = T[(p - 1) * 16 + l];
        if (SIGN > 0) w.y = -w.y;
        dst[p] = ddi_cmul(v[ddi_out16(p)], w);
    }
}
// pass 2 of lane p: reads A(l, p) over l, transforms; output X(p + 16 u) is left in v[ddi_out16(u)]
template <int SIGN>
__device__ __forceinline__ void ddi_fft256_pass2(double2 (&v)[16], const double2 *row, const int p) {
#pragma unroll
    for (int l = 0; l < 16; ++l) v[l] = row[17 * l + p];
    ddi_fft16<SIGN, false>(v);
}

// The a-pass kernels for rows of 512 real values (M = 256) in the transposed layout of the fused b-pass: a block of 256 threads takes 16
// consecutive ib of one slab, half a warp per row.  Forward: the 128 non-zero complex inputs z(j) = x(2j) + i x(2j+1) come straight from
// the spin array (pass 1 with half its inputs zero), the split X(k) = E(k) + W^k O(k) is done in place for the pair (k, 256 - k), and the
// rows leave through a transposed copy (16 consecutive ib = 256 contiguous bytes per wave number).
constexpr int DDI_A256_ROWS = 16, DDI_A256_WS = DDI_LP256 + 1;      // rows per block; row stride (X(256) has a slot of its own)
constexpr size_t DDI_A256_SMEM = ((size_t)DDI_A256_ROWS * DDI_A256_WS + 240) * sizeof(double2);
__global__ void __launch_bounds__(256, 3) ddi_apass256_fwd_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ n, int SL,
                                                               const double *__restrict__ mu_b, const double2 *__restrict__ tw,
                                                               cufftDoubleComplex *__restrict__ out) {
    extern __shared__ double2 ddi_sm[];
    constexpr int M = 256;
    double2 *T = ddi_sm + DDI_A256_ROWS * DDI_A256_WS;
    ddi_fill_t256(T, tw, threadIdx.x, blockDim.x);
    ddi_wait_upstream();
    const int hw = threadIdx.x >> 4, l = threadIdx.x & 15;                 // row of the block, lane of the half warp
    const unsigned hmask = 0xffffu << (threadIdx.x & 16);      // the lanes of this half warp
    const int rowid = blockIdx.x * DDI_A256_ROWS + hw;
    const int ib = rowid % L.Nb, slab = rowid / L.Nb;
    const int bc = slab / L.Nc, ic = slab - bc * L.Nc, sb = bc / 3, comp = bc - 3 * sb;
    const double mu = mu_b[sb];
    const double2 *src = (const double2 *)(n + (size_t)sb * L.sub + ((size_t)(ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + comp * L.PA + L.LA);
    double2 *row = ddi_sm + hw * DDI_A256_WS;
    double2 v[16];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = __ldg(src + l + 16 * q);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        double m0 = mu, m1 = mu;
        if (L.mu_ratio) { const double2 r = ddi_row_ratio(L, sb, ib, ic, l + 16 * q); m0 *= r.x; m1 *= r.y; }
        v[q].x *= m0; v[q].y *= m1;
    }
    __syncthreads();                                                       // T is complete
    ddi_fft256_pass1<-1, true>(v, row, T, l);
    __syncwarp(hmask);
    ddi_fft256_pass2<-1>(v, row, l);
    __syncwarp(hmask);                                                          // every lane has read the row
#pragma unroll
    for (int u = 0; u < 16; ++u) row[l + 17 * u] = v[ddi_out16(u)];        // Z(l + 16 u), natural order
    __syncwarp(hmask);
    // split in place: lane l takes k = l + 16 i, i < 8 (and lane 0 also k = 128), together with 256 - k
#pragma unroll
    for (int i = 0; i <= 8; ++i) {
        const int k = l + 16 * i;
        if (i == 8 && l != 0) break;
        const int km = (M - k) & (M - 1);
        const double2 zk = row[ddi_pad16(k)], zm = row[ddi_pad16(km)];
        const double er = 0.5 * (zk.x + zm.x), ei = 0.5 * (zk.y - zm.y);            // E = (Z(k) + conj Z(M-k)) / 2
        const double orr = 0.5 * (zk.y + zm.y), oi = -0.5 * (zk.x - zm.x);          // O = (Z(k) - conj Z(M-k)) / (2i)
        const double2 w = __ldg(tw + k);                                            // exp(-2 pi i k / 512)
        const double pr = fma(orr, w.x, -oi * w.y), pi = fma(orr, w.y, oi * w.x);   // W^k O
        row[ddi_pad16(k)] = make_double2(er + pr, ei + pi);                         // X(k) = E + W^k O
        row[ddi_pad16(M - k)] = make_double2(er - pr, -(ei - pi));                  // X(M - k) = conj(E - W^k O)
    }
    __syncthreads();
    const int ib0 = (blockIdx.x * DDI_A256_ROWS) % L.Nb;
    cufftDoubleComplex *o = out + (size_t)slab * L.Nb + ib0;
    for (int idx = threadIdx.x; idx < (M + 1) * DDI_A256_ROWS; idx += 256) {
        const int k = idx >> 4, w = idx & 15;
        o[(size_t)k * SL * L.Nb + w] = ddi_sm[w * DDI_A256_WS + ddi_pad16(k)];
    }
}

// inverse: the two partial results [r][ka][slab][ib] are added while they are gathered into the rows; Z(k) = E + i O is rebuilt in place
// for the pair (k, 256 - k); of the transform only the 128 outputs that are spins are stored (the rest is the zero padding's image).
__global__ void __launch_bounds__(256) ddi_apass256_inv_kernel(const __grid_constant__ DevicePlan L, const cufftDoubleComplex *__restrict__ in, int SL,
                                                               const double *__restrict__ mu_b, double scale0, const double2 *__restrict__ tw,
                                                               double *__restrict__ f, size_t part1) {
    extern __shared__ double2 ddi_sm[];
    constexpr int M = 256;
    double2 *T = ddi_sm + DDI_A256_ROWS * DDI_A256_WS;
    ddi_fill_t256(T, tw, threadIdx.x, blockDim.x);
    ddi_wait_upstream();
    const int hw = threadIdx.x >> 4, l = threadIdx.x & 15;
    const unsigned hmask = 0xffffu << (threadIdx.x & 16);      // the lanes of this half warp
    const int rowid = blockIdx.x * DDI_A256_ROWS + hw;
    const int ib = rowid % L.Nb, slab = rowid / L.Nb;
    const int bc = slab / L.Nc, ic = slab - bc * L.Nc, sb = bc / 3, comp = bc - 3 * sb;
    const double scale = mu_b[sb] * scale0;
    double2 *row = ddi_sm + hw * DDI_A256_WS;
    {
        const int ib0 = (blockIdx.x * DDI_A256_ROWS) % L.Nb;
        const cufftDoubleComplex *g0 = in + (size_t)slab * L.Nb + ib0, *g1 = g0 + part1;
        constexpr int total = M * DDI_A256_ROWS, U = 8;                   // wave numbers k < 256: 2 x 8 elements per thread ...
        double2 q0 = make_double2(0.0, 0.0), q1 = q0;                      // ... and k = 256: one element for the first 16 threads
        if (threadIdx.x < DDI_A256_ROWS) {
            const size_t o = (size_t)M * SL * L.Nb + threadIdx.x;
            q0 = __ldg(g0 + o); q1 = __ldg(g1 + o);
        }
        for (int base = threadIdx.x; base < total; base += U * 256) {
            double2 p0[U], p1[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int idx = base + u * 256;
                const size_t o = (size_t)(idx >> 4) * SL * L.Nb + (idx & 15);
                p0[u] = __ldg(g0 + o); p1[u] = __ldg(g1 + o);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int idx = base + u * 256;
                ddi_sm[(idx & 15) * DDI_A256_WS + ddi_pad16(idx >> 4)] = make_double2(p0[u].x + p1[u].x, p0[u].y + p1[u].y);
            }
        }
        if (threadIdx.x < DDI_A256_ROWS) ddi_sm[threadIdx.x * DDI_A256_WS + ddi_pad16(M)] = make_double2(q0.x + q1.x, q0.y + q1.y);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i <= 8; ++i) {
        const int k = l + 16 * i;
        if (i == 8 && l != 0) break;
        const double2 xk = row[ddi_pad16(k)], xm = row[ddi_pad16(M - k)];
        const double er = xk.x + xm.x, ei = xk.y - xm.y;                            // E = X(k) + conj X(M-k)
        const double dr = xk.x - xm.x, di = xk.y + xm.y;                            // X(k) - conj X(M-k)
        const double2 w = __ldg(tw + k);                                            // times exp(+2 pi i k / 512)
        const double orr = fma(dr, w.x, di * w.y), oi = fma(di, w.x, -dr * w.y);
        row[ddi_pad16(k)] = make_double2(er - oi, ei + orr);                        // Z(k) = E + i O
        if (k) row[ddi_pad16(M - k)] = make_double2(er + oi, -(ei - orr));          // Z(M - k) = conj(E - i O)
    }
    __syncwarp(hmask);
    double2 v[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) v[q] = row[l + 17 * q];
    __syncwarp(hmask);
    ddi_fft256_pass1<+1, false>(v, row, T, l);
    __syncwarp(hmask);
    ddi_fft256_pass2<+1>(v, row, l);
    double2 *dst = (double2 *)(f + (size_t)sb * L.sub + ((size_t)(ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + comp * L.PA + L.LA);
#pragma unroll
    for (int u = 0; u < 8; ++u) {                                                   // z(j), j = l + 16 u < 128
        const int j = l + 16 * u;
        const double2 z = v[ddi_out16(u)];
        double m0 = scale, m1 = scale;
        if (L.mu_ratio) { const double2 r = ddi_row_ratio(L, sb, ib, ic, j); m0 *= r.x; m1 *= r.y; }
        dst[j] = make_double2(m0 * z.x, m1 * z.y);
    }
}

// Slab path, the transform along c fused with the tensor contraction, per in-plane wave vector q = (kx, ky):
//   M^(kz) = sum_{z < NZ} M2(z) w^(kz z),  w = exp(-2 pi i / PZ)     (pruned: planes z >= NZ are zero padding)
//   H^(kz) = K^(kz) . M^(kz)                                          (6-component real symmetric tensor)
//   H2(z)  = sum_{kz < PZ} H^(kz) w^(-kz z),  z < NZ only
// Two threads share a column: thread e of the pair takes the wave numbers kz = 2 j + e,
//   M^(2 j + e) = sum_z [M2(z) w^(e z)] W_NZ^(j z),    H2(z) = sum_e w^(-e z) sum_j H^(2 j + e) W_NZ^(-j z),
// i.e. a length-NZ transform of the (for e = 1: pre-twisted) column, the contraction at its own NZ wave numbers, the inverse length-NZ
// transform and the twist back; the two halves are added through shared memory.  Each thread then holds 3 NZ complex numbers instead of
// the 3 (NZ + PZ) of a one-thread-per-column kernel (255 registers, 12.5 % occupancy in round 1).  A mirror-symmetric tensor
// (K(PZ - kz) = +-K(kz), ddi_mirror_check_kernel) is read once for kz and PZ - kz, which have the same parity and so the same thread.
// PAD = false: a single plane that is not padded along c (NZ = PZ = 1): no transform at all, thread e = 1 idles.
// M2 / H2: element (kb, slab = c NZ + z, ka) at (kb SL + slab) S1p + ka, S1p the row pitch (H2 may be M2: every column is read, then
// written, by its own pair of threads); Kre: [6][PZ][S2] with q = kb S1 + ka.
// The work of thread e on its column x (3 components x NZ planes, complex): twist, forward transform, contraction at its NZ wave numbers
// with the tensor planes that kload(plane, k[6]) delivers (xx, xy, xz, yy, yz, zz), inverse transform, twist back.  In place.
template <int NZ, bool PAD, bool MIRROR, class KLoad>
__device__ __forceinline__ void ddi_column_half(double (&xr)[3][NZ], double (&xi)[3][NZ], const int e, KLoad &&kload) {
    constexpr int PZ = PAD ? 2 * NZ : NZ;
    // contraction at one wave number; position p of the transformed column holds kz = 2 ddi_pos(p) + e
    auto contract = [&](const int p, const double kxx, const double kxy, const double kxz, const double kyy, const double kyz, const double kzz) {
        const double r0 = xr[0][p], r1 = xr[1][p], r2 = xr[2][p], i0 = xi[0][p], i1 = xi[1][p], i2 = xi[2][p];
        xr[0][p] = kxx * r0 + kxy * r1 + kxz * r2; xr[1][p] = kxy * r0 + kyy * r1 + kyz * r2; xr[2][p] = kxz * r0 + kyz * r1 + kzz * r2;
        xi[0][p] = kxx * i0 + kxy * i1 + kxz * i2; xi[1][p] = kxy * i0 + kyy * i1 + kyz * i2; xi[2][p] = kxz * i0 + kyz * i1 + kzz * i2;
    };
    // (the parity is the outermost branch -- uniform per warp in every caller -- so that the loads of the first tensor planes, which
    // depend on it, can be issued before the transform and overlap it)
    auto work = [&](auto ec) {
        constexpr int E = decltype(ec)::value;
        // planes this thread reads: kz = 2 j + E, j < NJ (MIRROR: up to PZ / 2 only, the rest are mirror images); the tensor of plane
        // j + AHEAD is loaded before plane j is contracted
        constexpr int NJ = !PAD ? 1 : (MIRROR ? (PZ / 2 - E) / 2 + 1 : NZ);
        constexpr int AHEAD = 2;
        double k[AHEAD + 1][6];
#pragma unroll
        for (int j = 0; j < AHEAD && j < NJ; ++j) kload(PAD ? 2 * j + E : 0, k[j]);
        if constexpr (PAD) {
            if constexpr (E == 1) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int z = 1; z < NZ; ++z) {
                        if constexpr (ddi_pow2(NZ)) ddi_rot16(z * (16 / PZ), xr[c][z], xi[c][z]);
                        else {
                            const double wr = DDI_TWR[PZ][z], wi = DDI_TWI[PZ][z], r = xr[c][z], i = xi[c][z];
                            xr[c][z] = fma(r, wr, -i * wi); xi[c][z] = fma(r, wi, i * wr);
                        }
                    }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) ddi_dft_fwd<NZ>(xr[c], xi[c]);
        }
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int kz = PAD ? 2 * j + E : 0;
            if (j + AHEAD < NJ) kload(kz + 2 * AHEAD, k[(j + AHEAD) % (AHEAD + 1)]);
            const double(&kk)[6] = k[j % (AHEAD + 1)];
            contract(ddi_pos<NZ>(j), kk[0], kk[1], kk[2], kk[3], kk[4], kk[5]);
            if (MIRROR && kz > 0 && 2 * kz < PZ)                        // plane PZ - kz: the same values, xz and yz with the opposite sign
                contract(ddi_pos<NZ>((PZ - kz - E) / 2), kk[0], kk[1], -kk[2], kk[3], -kk[4], kk[5]);
        }
        if constexpr (PAD) {
#pragma unroll
            for (int c = 0; c < 3; ++c) ddi_dft_inv<NZ>(xr[c], xi[c]);
            if constexpr (E == 1) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int z = 1; z < NZ; ++z) {
                        if constexpr (ddi_pow2(NZ)) ddi_rot16(16 - z * (16 / PZ), xr[c][z], xi[c][z]);
                        else {
                            const double wr = DDI_TWR[PZ][z], wi = -DDI_TWI[PZ][z], r = xr[c][z], i = xi[c][z];
                            xr[c][z] = fma(r, wr, -i * wi); xi[c][z] = fma(r, wi, i * wr);
                        }
                    }
            }
        }
    };
    if (e) work(spin_ddi_int<1>{}); else work(spin_ddi_int<0>{});
}

constexpr int DDI_CT_COLS = 64;      // columns per block: 2 x 64 threads
template <int NZ, bool PAD, bool MIRROR>
__global__ void __launch_bounds__(2 * DDI_CT_COLS, 4) ddi_slab_contract_kernel(const double *__restrict__ Kre, const cufftDoubleComplex *__restrict__ M2,
                                                                             cufftDoubleComplex *H2, long long S2, int S1, int S1p) {
    constexpr int PZ = PAD ? 2 * NZ : NZ;
    static_assert(PAD || NZ == 1, "only a single plane goes unpadded");
    __shared__ double2 half1[3 * NZ][DDI_CT_COLS];
    const int lane_col = threadIdx.x % DDI_CT_COLS, e = threadIdx.x / DDI_CT_COLS;
    const long long q = (long long)blockIdx.x * DDI_CT_COLS + lane_col;
    const bool live = q < S2 && (PAD || e == 0);
    const long long kb = live ? q / S1 : 0, ka = live ? q - kb * S1 : 0;
    const size_t col = (size_t)kb * (3 * NZ) * S1p + ka;           // slab 0 of this wave vector; slabs are one row pitch apart
    double xr[3][NZ], xi[3][NZ];
    if (live) {
        // the tensor planes of this thread are needed only after the forward transform, when no registers are left to hold them: ask L2
        // for their lines now (one line per 16 threads), so that the loads below the transform find them there
        if ((lane_col & 15) == 0) {
#pragma unroll
            for (int j = 0; j < NZ; ++j) {
                const int kz = PAD ? 2 * j + e : 0;
                if (MIRROR && 2 * kz > PZ) continue;
#pragma unroll
                for (int m = 0; m < 6; ++m) asm volatile("prefetch.global.L2 [%0];" ::"l"(Kre + ((size_t)m * PZ + kz) * S2 + q));
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int z = 0; z < NZ; ++z) {
                const cufftDoubleComplex v = M2[col + (size_t)(c * NZ + z) * S1p];
                xr[c][z] = v.x; xi[c][z] = v.y;
            }
        const size_t st = (size_t)PZ * S2;
        ddi_column_half<NZ, PAD, MIRROR>(xr, xi, e, [&](const int kz, double (&k)[6]) {
            const size_t o = (size_t)kz * S2 + q;
#pragma unroll
            for (int m = 0; m < 6; ++m) k[m] = Kre[m * st + o];
        });
        if constexpr (PAD) {
            if (e) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int z = 0; z < NZ; ++z) half1[c * NZ + z][lane_col] = make_double2(xr[c][z], xi[c][z]);
            }
        }
    }
    if constexpr (PAD) __syncthreads();
    if (live && e == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int z = 0; z < NZ; ++z) {
                double r = xr[c][z], i = xi[c][z];
                if constexpr (PAD) { const double2 h = half1[c * NZ + z][lane_col]; r += h.x; i += h.y; }
                H2[col + (size_t)(c * NZ + z) * S1p] = make_cuDoubleComplex(r, i);
            }
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// Fused b-pass (round 2; one basis atom, rows and columns of power-of-two length): forward transform along b, transform along c,
// tensor contraction, inverse transform along c and inverse transform along b in ONE kernel, so that the full spectra (2 x 50 MB per
// pass on cfg5) never exist in HBM.  The column of length P1 = 2 Nb has Nb occupied rows followed by Nb zeros, and only Nb rows of the
// result are needed, so the wave numbers kb split by parity r:
//     X(2 k' + r) = sum_{ib < Nb} [x(ib) W^(r ib)] W_Nb^(k' ib),        y(ib) = sum_r W^(-r ib) sum_k' Y(2 k' + r) W_Nb^(-k' ib),   W = exp(-2 pi i / P1):
// two independent transforms of length Nb.  A block takes one ka and one parity r: it reads its 3 NZ columns of Nb rows (contiguous in the
// [ka][slab][ib] layout the a-pass kernels write in this mode), transforms them (one warp per column, Stockham passes in place; the first pass
// reads global memory and applies the twist), contracts every wave
// vector (ka, kb = 2 k' + r) along c exactly like ddi_slab_contract_kernel (two threads per column, tensor from a copy laid out
// [ka][r][component][plane][k'] when the plan is built), transforms back and writes its partial result; the inverse a-pass adds the two
// parities.  (Measured slower: one block per ka taking the two parities in turn and adding them itself, 76 instead of 66 us; the two
// parities as a cluster of two blocks that add their results through distributed shared memory and write one array, 66.8 instead of
// 58.2 us -- the inverse a-pass gains 3 us from the halved input, the fused kernel loses 8.6 to the cluster barriers and the extra pass.)  Shared memory: 3 NZ padded columns of Nb complex numbers (cfg5: 24 columns x 4.6 KB = 110.6 KB, two blocks of 256 threads per SM,
// so that one block's loads overlap the other's arithmetic).
constexpr int DDI_BF_THREADS = 256, DDI_BF_WARPS = DDI_BF_THREADS / 32;
// F256: columns of length 256 -- half a warp per column, two passes of radix 16 (ddi_fft256_pass1 / 2), rows padded by one in 16.
// PAD = false: a single plane that is not padded along c (a monolayer, NZ = PZ = 1): no transform along c, one thread per wave vector.
template <int NZ, bool MIRROR, bool F256, bool PAD = true>
__global__ void __launch_bounds__(DDI_BF_THREADS, 2) ddi_bfused_kernel(const double *__restrict__ Kb, const double2 *__restrict__ Tin, double2 *__restrict__ Tout,
                                                                        const int lgM_, const int S1, const double2 *__restrict__ tw) {
    constexpr int SL = 3 * NZ, NPL = !PAD ? 1 : (MIRROR ? NZ + 1 : 2 * NZ), PADSH = F256 ? 4 : 3;
    static_assert(PAD || (NZ == 1 && !MIRROR), "only a single plane goes unpadded");
    extern __shared__ double2 ddi_sm[];
    const int lgM = F256 ? 8 : lgM_;
    const int M = 1 << lgM, LP = M + (M >> PADSH);
    auto pad = [](const int i) { return i + (i >> PADSH); };
    const int ka = blockIdx.x >> 1, r = blockIdx.x & 1;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const double *Kme = Kb + (((size_t)ka * 2 + r) * 6 * NPL << lgM);
    // ask L2 for this block's tensor planes while the columns are transformed
    for (size_t i = (size_t)tid * 16; i < ((size_t)6 * NPL << lgM); i += (size_t)DDI_BF_THREADS * 16) asm volatile("prefetch.global.L2 [%0];" ::"l"(Kme + i));
    // the first M entries of the twiddle table, in shared memory behind the columns (all a pass or the twist ever reads)
    double2 *tws = ddi_sm + (size_t)SL * LP;
    for (int i = tid; i < M; i += DDI_BF_THREADS) tws[i] = __ldg(tw + i);
    if constexpr (F256) {
        // ---- forward, length 256: half a warp per column; pass 1 reads global memory (16 loads per lane in flight) and applies the twist
        double2 *T = tws + M;
        ddi_fill_t256(T, tw, tid, DDI_BF_THREADS);
        ddi_wait_upstream();
        __syncthreads();                                                       // tws and T are complete
        const int l = tid & 15;
        const unsigned hmask = 0xffffu << (tid & 16);      // the lanes of this half warp (the other half may have no column)
        for (int slab = tid >> 4; slab < SL; slab += DDI_BF_THREADS / 16) {
            const double2 *src = Tin + (((size_t)ka * SL + slab) << 8) + l;
            double2 *row = ddi_sm + slab * LP;
            double2 v[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) v[q] = __ldg(src + 16 * q);
            if (r) {
#pragma unroll
                for (int q = 0; q < 16; ++q) v[q] = ddi_cmul(v[q], tws[l + 16 * q]);
            }
            ddi_fft256_pass1<-1, false>(v, row, T, l);
            __syncwarp(hmask);
            ddi_fft256_pass2<-1>(v, row, l);
            __syncwarp(hmask);
#pragma unroll
            for (int u = 0; u < 16; ++u) row[l + 17 * u] = v[ddi_out16(u)];
        }
    } else {
    // ---- forward: one warp per column, in place in the column's shared-memory row (every lane holds its M / 32 elements between the
    // loads and the stores of a pass).  The first pass (always radix 8) reads global memory and applies the twist of the odd wave
    // numbers; the loads of the warp's next column are in flight while it transforms the current one.
        constexpr int NIT = (SL + DDI_BF_WARPS - 1) / DDI_BF_WARPS;
        const int span = M >> 3, j = min(lane, span - 1);
        double2 buf[2][8];
        auto fetch = [&](const int slab, double2 (&v)[8]) {
            const double2 *src = Tin + (((size_t)ka * SL + slab) << lgM) + j;
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = __ldg(src + q * span);
        };
        ddi_wait_upstream();
        if (warp < SL) fetch(warp, buf[0]);
        __syncthreads();                                                       // tws is complete
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int slab = warp + it * DDI_BF_WARPS;
            if (it + 1 < NIT && slab + DDI_BF_WARPS < SL) fetch(slab + DDI_BF_WARPS, buf[(it + 1) & 1]);
            if (slab < SL) {
                double2(&v)[8] = buf[it & 1];
                double2 *row = ddi_sm + (size_t)slab * LP;
                auto st = [&](int i, const double2 x) { row[ddi_pad(i)] = x; };
                if (r) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) v[q] = ddi_cmul(v[q], tws[j + q * span]);
                }
                if (lane < span) ddi_fft_finish<-1, 8>(v, lane, 0, lgM - 2, tws, st);
                for (int lgNs = 3; lgNs < lgM;) {
                    __syncwarp();
                    lgNs += ddi_fft_next_pass<-1, true>(lgM, lgNs, tws, lane, [&](int i) { return row[ddi_pad(i)]; }, st);
                }
            }
        }
    }
    __syncthreads();
    // ---- contraction along c: thread (k', e) of a round takes the wave numbers kz = 2 j + e of the wave vector (ka, kb = 2 k' + r)
    constexpr int half = DDI_BF_THREADS / 2;
    const int e = tid / half;
    if constexpr (!PAD) {
        for (int kp = tid; kp < M; kp += DDI_BF_THREADS) {
            double2 *col = ddi_sm + pad(kp);
            double k[6];
#pragma unroll
            for (int m = 0; m < 6; ++m) k[m] = __ldg(Kme + ((size_t)m << lgM) + kp);
            const double2 x = col[0], y = col[LP], z = col[2 * LP];
            col[0] = make_double2(k[0] * x.x + k[1] * y.x + k[2] * z.x, k[0] * x.y + k[1] * y.y + k[2] * z.y);
            col[LP] = make_double2(k[1] * x.x + k[3] * y.x + k[4] * z.x, k[1] * x.y + k[3] * y.y + k[4] * z.y);
            col[2 * LP] = make_double2(k[2] * x.x + k[4] * y.x + k[5] * z.x, k[2] * x.y + k[4] * y.y + k[5] * z.y);
        }
    } else
    for (int k0 = 0; k0 < M; k0 += half) {
        const int kp = k0 + (tid - e * half);
        const bool live = kp < M;
        double2 *col = ddi_sm + pad(kp);
        double xr[3][NZ], xi[3][NZ];
        if (live) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int z = 0; z < NZ; ++z) { const double2 v = col[(size_t)(c * NZ + z) * LP]; xr[c][z] = v.x; xi[c][z] = v.y; }
            ddi_column_half<NZ, PAD, MIRROR>(xr, xi, e, [&](const int kz, double (&k)[6]) {
#pragma unroll
                for (int m = 0; m < 6; ++m) k[m] = __ldg(Kme + ((size_t)(m * NPL + kz) << lgM) + kp);
            });
        }
        __syncthreads();                                                      // both halves have read the column
        if (live && e) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int z = 0; z < NZ; ++z) col[(size_t)(c * NZ + z) * LP] = make_double2(xr[c][z], xi[c][z]);
        }
        __syncthreads();
        if (live && !e) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int z = 0; z < NZ; ++z) {
                    double2 *q = col + (size_t)(c * NZ + z) * LP;
                    const double2 h = *q;
                    *q = make_double2(xr[c][z] + h.x, xi[c][z] + h.y);
                }
        }
    }
    __syncthreads();
    if constexpr (F256) {
        // ---- inverse, length 256: the outputs of pass 2 go straight to global memory (twisted back), 256 contiguous bytes per half warp
        const double2 *T = tws + M;
        const int l = tid & 15;
        const unsigned hmask = 0xffffu << (tid & 16);
        for (int slab = tid >> 4; slab < SL; slab += DDI_BF_THREADS / 16) {
            double2 *dstg = Tout + ((((size_t)r * S1 + ka) * SL + slab) << 8) + l;
            double2 *row = ddi_sm + slab * LP;
            double2 v[16];
#pragma unroll
            for (int q = 0; q < 16; ++q) v[q] = row[l + 17 * q];
            __syncwarp(hmask);
            ddi_fft256_pass1<+1, false>(v, row, T, l);
            __syncwarp(hmask);
            ddi_fft256_pass2<+1>(v, row, l);
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                double2 x = v[ddi_out16(u)];
                if (r) { double2 w = tws[l + 16 * u]; w.y = -w.y; x = ddi_cmul(x, w); }
                dstg[16 * u] = x;
            }
        }
    } else {
    // ---- inverse: one warp per column, the last pass writes the partial result of this parity (twisted back) to global memory
    for (int slab = warp; slab < SL; slab += DDI_BF_WARPS) {
        double2 *dstg = Tout + ((((size_t)r * S1 + ka) * SL + slab) << lgM);
        double2 *row = ddi_sm + (size_t)slab * LP;
        auto ld = [&](int i) { return row[ddi_pad(i)]; };
        int lgNs = 0;
        while (lgM - lgNs > 3) {
            lgNs += ddi_fft_next_pass<+1, true>(lgM, lgNs, tws, lane, ld, [&](int i, const double2 v) { row[ddi_pad(i)] = v; });
            __syncwarp();
        }
        ddi_fft_next_pass<+1, false>(lgM, lgNs, tws, lane, ld, [&](int i, double2 v) {
            if (r) { double2 w = tws[i]; w.y = -w.y; v = ddi_cmul(v, w); }
            dstg[i] = v;
        });
    }
    }
}

// the tensor in the order ddi_bfused_kernel reads it: Kb[ka][r][component][plane][k'] = Kre[component][plane][kb = 2 k' + r][ka]
__global__ void ddi_bfused_tensor_kernel(const double *__restrict__ Kre, double *__restrict__ Kb, int PZ, int NPL, int M, int S1) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)S1 * 2 * 6 * NPL * M;
    if (i >= total) return;
    const int kp = (int)(i % M);
    long long t = i / M;
    const int m = (int)(t % NPL); t /= NPL;
    const int comp = (int)(t % 6); t /= 6;
    const int r = (int)(t % 2);
    const int ka = (int)(t / 2);
    const long long S2 = (long long)(2 * M) * S1;
    Kb[i] = Kre[((long long)comp * PZ + m) * S2 + (long long)(2 * kp + r) * S1 + ka];
}

// The same for several basis atoms ("one FFT per sublattice + inter-sublattice convolutions"): H_a^(kz) = sum_b K_ab^(kz) . M_b^(kz)
// with COMPLEX tensor spectra (K_ab(-Delta) = K_ba(Delta): only the diagonal blocks are even), read from the 3-D half spectrum
// Khat[a][b][6][PZ][S2].  blockIdx.y = target sublattice a; the thread transforms the column of every source sublattice b in turn and
// accumulates the contracted spectrum, then transforms back.  Out of place (M2 is read by every a): slabs are (b 3 + c) NZ + z.
template <int NZ, bool PAD>
__global__ void __launch_bounds__(2 * DDI_CT_COLS) ddi_slab_contract_mb_kernel(const cufftDoubleComplex *__restrict__ Khat, const cufftDoubleComplex *__restrict__ M2,
                                                                                cufftDoubleComplex *__restrict__ H2, int nb, long long S2, int S1, int S1p) {
    constexpr int PZ = PAD ? 2 * NZ : NZ;
    static_assert(PAD || NZ == 1, "only a single plane goes unpadded");
    __shared__ double2 half1[3 * NZ][DDI_CT_COLS];
    const int lane_col = threadIdx.x % DDI_CT_COLS, e = threadIdx.x / DDI_CT_COLS, a = blockIdx.y;
    const long long q = (long long)blockIdx.x * DDI_CT_COLS + lane_col;
    const bool live = q < S2 && (PAD || e == 0);
    const long long kb = live ? q / S1 : 0, ka = live ? q - kb * S1 : 0;
    const size_t SLr = (size_t)nb * 3 * NZ;
    const size_t col = (size_t)kb * SLr * S1p + ka;                // slab 0 of this wave vector
    const size_t Ph = (size_t)PZ * S2;                             // points of one tensor component
    double hr[3][NZ], hi[3][NZ];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int z = 0; z < NZ; ++z) { hr[c][z] = 0.0; hi[c][z] = 0.0; }
    if (live) {
        for (int b = 0; b < nb; ++b) {
            double xr[3][NZ], xi[3][NZ];
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int z = 0; z < NZ; ++z) {
                    const cufftDoubleComplex v = M2[col + (size_t)((b * 3 + c) * NZ + z) * S1p];
                    xr[c][z] = v.x; xi[c][z] = v.y;
                }
            if constexpr (PAD) {
                if (e) {
#pragma unroll
                    for (int c = 0; c < 3; ++c)
#pragma unroll
                        for (int z = 1; z < NZ; ++z) {
                            const double wr = DDI_TWR[PZ][z], wi = DDI_TWI[PZ][z], r = xr[c][z], i = xi[c][z];
                            xr[c][z] = fma(r, wr, -i * wi); xi[c][z] = fma(r, wi, i * wr);
                        }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) ddi_dft_fwd<NZ>(xr[c], xi[c]);
            }
            const cufftDoubleComplex *K = Khat + (size_t)(a * nb + b) * 6 * Ph + q;
            auto planes = [&](auto ec) {
                constexpr int E = decltype(ec)::value;
#pragma unroll
                for (int j = 0; j < NZ; ++j) {
                    const int kz = PAD ? 2 * j + E : 0, p = ddi_pos<NZ>(j);
                    const size_t o = (size_t)kz * S2;
                    const cufftDoubleComplex kxx = K[o], kxy = K[Ph + o], kxz = K[2 * Ph + o], kyy = K[3 * Ph + o], kyz = K[4 * Ph + o], kzz = K[5 * Ph + o];
                    const double r0 = xr[0][p], r1 = xr[1][p], r2 = xr[2][p], i0 = xi[0][p], i1 = xi[1][p], i2 = xi[2][p];
                    // complex (k . m): re = k.x m.x - k.y m.y, im = k.x m.y + k.y m.x
                    hr[0][p] += kxx.x * r0 - kxx.y * i0 + kxy.x * r1 - kxy.y * i1 + kxz.x * r2 - kxz.y * i2;
                    hi[0][p] += kxx.x * i0 + kxx.y * r0 + kxy.x * i1 + kxy.y * r1 + kxz.x * i2 + kxz.y * r2;
                    hr[1][p] += kxy.x * r0 - kxy.y * i0 + kyy.x * r1 - kyy.y * i1 + kyz.x * r2 - kyz.y * i2;
                    hi[1][p] += kxy.x * i0 + kxy.y * r0 + kyy.x * i1 + kyy.y * r1 + kyz.x * i2 + kyz.y * r2;
                    hr[2][p] += kxz.x * r0 - kxz.y * i0 + kyz.x * r1 - kyz.y * i1 + kzz.x * r2 - kzz.y * i2;
                    hi[2][p] += kxz.x * i0 + kxz.y * r0 + kyz.x * i1 + kyz.y * r1 + kzz.x * i2 + kzz.y * r2;
                }
            };
            if (e) planes(spin_ddi_int<1>{}); else planes(spin_ddi_int<0>{});
        }
        if constexpr (PAD) {
#pragma unroll
            for (int c = 0; c < 3; ++c) ddi_dft_inv<NZ>(hr[c], hi[c]);
            if (e) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int z = 0; z < NZ; ++z) {
                        double r = hr[c][z], i = hi[c][z];
                        if (z > 0) { const double wr = DDI_TWR[PZ][z], wi = -DDI_TWI[PZ][z]; const double t = fma(r, wr, -i * wi); i = fma(r, wi, i * wr); r = t; }
                        half1[c * NZ + z][lane_col] = make_double2(r, i);
                    }
            }
        }
    }
    if constexpr (PAD) __syncthreads();
    if (live && e == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int z = 0; z < NZ; ++z) {
                double r = hr[c][z], i = hi[c][z];
                if constexpr (PAD) { const double2 h = half1[c * NZ + z][lane_col]; r += h.x; i += h.y; }
                H2[col + (size_t)((a * 3 + c) * NZ + z) * S1p] = make_cuDoubleComplex(r, i);
            }
    }
}

// Is the tensor spectrum mirror symmetric along c, K_ab(kz) = s_ab K_ab(PZ - kz) with s = -1 for xz, yz and +1 otherwise?  (True when c is
// perpendicular to a and b.)  out[0] = max |K(kz) - s K(PZ - kz)|, out[1] = max |K| as the bit patterns of non-negative doubles,
// which order like unsigned integers.
__global__ void ddi_mirror_check_kernel(const double *__restrict__ Kre, int PZ, long long S2, unsigned long long *out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double dev = 0.0, mag = 0.0;
    if (i < 6LL * PZ * S2) {
        const int comp = (int)(i / ((long long)PZ * S2));
        const long long r = i - (long long)comp * PZ * S2;
        const int kz = (int)(r / S2);
        const long long q = r - (long long)kz * S2;
        const double sgn = (comp == 2 || comp == 4) ? -1.0 : 1.0;
        const double a = Kre[i], b = Kre[((long long)comp * PZ + (PZ - kz) % PZ) * S2 + q];
        dev = fabs(a - sgn * b); mag = fabs(a);
    }
    for (int o = 16; o > 0; o >>= 1) {
        dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
        mag = fmax(mag, __shfl_xor_sync(0xffffffffu, mag, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(out, (unsigned long long)__double_as_longlong(dev));
        atomicMax(out + 1, (unsigned long long)__double_as_longlong(mag));
    }
}

#define SPIN_FFT(call)                                                                                         \
    do {                                                                                                       \
        cufftResult r__ = (call);                                                                              \
        if (r__ != CUFFT_SUCCESS) return spin::fail(SPIN_ERR_CUDA, "%s failed: cufft error %d (%s:%d)", #call, \
                                                    (int)r__, __FILE__, __LINE__);                             \
    } while (0)

}  // namespace

// a kernel of the fused path, launched with programmatic stream serialisation (option use_pdl = 0: the plain way); see ddi_wait_upstream
template <class... KArgs, class... Args>
static cudaError_t ddi_launch(const spin_system *s, void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, Args &&...args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid, 1, 1); cfg.blockDim = dim3(block, 1, 1); cfg.dynamicSmemBytes = smem; cfg.stream = s->stream;
    cudaLaunchAttribute at;
    memset(&at, 0, sizeof(at));
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;
    if (s->opt_pdl != 0) { cfg.attrs = &at; cfg.numAttrs = 1; }
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

bool spin::ddi_graph_ok(const spin_system *s) { return s->ddi && s->ddi->fused_b; }

const char *spin::ddi_path_name(const spin_system *s) {
    const DdiState *d = s->ddi;
    if (!s->ddi_on || !d) return "off";
    if (!d->slab) return "3d";
    if (d->fused_b) return d->mirror ? "slab+mirror+own-a+fused-b" : "slab+own-a+fused-b";
    if (d->own_a) return d->mirror ? "slab+mirror+own-a" : "slab+own-a";
    return d->mirror ? "slab+mirror" : "slab";
}

void spin::ddi_release(spin_system *s) {
    DdiState *d = s->ddi;
    if (!d) return;
    if (d->have_plans) { cufftDestroy(d->plan_r2c); cufftDestroy(d->plan_c2r); }
    if (d->slab) {
        if (d->plan_a_fwd) cufftDestroy(d->plan_a_fwd);
        if (d->plan_a_inv) cufftDestroy(d->plan_a_inv);
        if (d->plan_b) cufftDestroy(d->plan_b);
    }
    cudaFree(d->s_in); cudaFree(d->s_out); cudaFree(d->s_a); cudaFree(d->s_b); cudaFree(d->s_c); cudaFree(d->s_d);
    cudaFree(d->d_Kre); cudaFree(d->d_tw); cudaFree(d->d_tw_b); cudaFree(d->d_Kb);
    cudaFree(d->d_Mpad); cudaFree(d->d_Hpad); cudaFree(d->d_Mhat); cudaFree(d->d_Hhat); cudaFree(d->d_Khat); cudaFree(d->d_geom);
    delete d;
    s->ddi = nullptr;
}

int spin::ddi_prepare(spin_system *s) {
    ddi_release(s);
    DdiState *d = new DdiState();
    memset(d, 0, sizeof(*d));
    s->ddi = d;
    const int nb = s->nb;
    d->rank = 0;
    for (int k = 0; k < 3; ++k) d->P[k] = (s->nc[k] > 1) ? 2 * s->nc[k] : 1;
    d->Ptot = (int64_t)d->P[0] * d->P[1] * d->P[2];
    // cuFFT dims slowest first, unit dims dropped (they do not change the strides)
    for (int k = 2; k >= 0; --k) if (d->P[k] > 1) d->fdims[d->rank++] = d->P[k];
    d->Phalf = d->Ptot;
    if (d->rank > 0) { const int inner = d->fdims[d->rank - 1]; d->Phalf = d->Ptot / inner * (inner / 2 + 1); }
    // slab path: both in-plane directions padded, at most 8 planes along c
    d->NZ = s->nc[2]; d->PZ = d->P[2];
    d->R2 = (int64_t)d->P[0] * d->P[1]; d->S2 = (int64_t)d->P[1] * (d->P[0] / 2 + 1);
    // several basis atoms: complex tensor spectra per sublattice pair, up to 4 planes (the contraction holds two columns in registers)
    const bool want_slab = s->opt_ddi_slab && d->P[0] > 1 && d->P[1] > 1 && d->NZ <= (nb == 1 ? 8 : 4);
    size_t nreal = (size_t)nb * 3 * d->Ptot, ncplx = (size_t)nb * 3 * d->Phalf;
    d->SL = 3 * d->NZ * nb; d->S1 = d->P[0] / 2 + 1; d->S1p = d->S1;      // a 128-byte row pitch (264) was measured slower: 368 vs 347 us per step on cfg5
    // own a-pass: rows of power-of-two length, 8 <= Na <= 2048 (option ddi_slab = 2 keeps cuFFT's, for comparison)
    const int Na = s->nc[0];
    d->own_a = want_slab && s->opt_ddi_slab != 2 && Na >= 8 && Na <= 2048 && (Na & (Na - 1)) == 0;
    // fused b-pass: one basis atom, power-of-two columns too, padded along c, and the block's columns fit into shared memory
    // (option ddi_slab = 3 keeps cuFFT's b-pass and the separate contraction, for comparison)
    const int Nb_ = s->nc[1];
    d->bf_smem = ((size_t)(3 * d->NZ) * (size_t)(Nb_ + Nb_ / 8) + (size_t)Nb_) * sizeof(double2);      // columns + twiddles
    if (Nb_ == 256) d->bf_smem = ((size_t)(3 * d->NZ) * DDI_LP256 + 256 + 240) * sizeof(double2);         // columns (padded by 1 in 16) + twiddles + pass-1 table
    d->fused_b = d->own_a && s->opt_ddi_slab == 1 && nb == 1 && Nb_ >= 8 && Nb_ <= 256 && (Nb_ & (Nb_ - 1)) == 0 && (d->PZ == 2 * d->NZ || d->PZ == 1) && d->bf_smem <= 220 * 1024;
    if (want_slab) {
        const size_t nr = (size_t)s->nc[1] * d->SL * d->P[0], nc_ = (size_t)d->P[1] * d->SL * d->S1p;
        if (!d->own_a) {
            SPIN_CUDA(cudaMalloc(&d->s_in, nr * sizeof(double)));
            SPIN_CUDA(cudaMalloc(&d->s_out, nr * sizeof(double)));
            SPIN_CUDA(cudaMemsetAsync(d->s_in, 0, nr * sizeof(double), s->stream));                // ia >= Na: zero padding, never written
        }
        SPIN_CUDA(cudaMalloc(&d->s_a, nc_ * sizeof(cufftDoubleComplex)));                          // (fused b-pass: half of it is used)
        SPIN_CUDA(cudaMalloc(&d->s_d, nc_ * sizeof(cufftDoubleComplex)));
        if (!d->fused_b) SPIN_CUDA(cudaMalloc(&d->s_b, nc_ * sizeof(cufftDoubleComplex)));
        if (nb > 1) SPIN_CUDA(cudaMalloc(&d->s_c, nc_ * sizeof(cufftDoubleComplex)));      // the contraction of several sublattices is out of place
        SPIN_CUDA(cudaMemsetAsync(d->s_a, 0, nc_ * sizeof(cufftDoubleComplex), s->stream));        // rows >= Nb: zero padding, never written
        nreal = 1; ncplx = 1;      // the buffers of the general path are not needed
    }
    SPIN_CUDA(cudaMalloc(&d->d_Mpad, nreal * sizeof(double)));
    SPIN_CUDA(cudaMalloc(&d->d_Hpad, nreal * sizeof(double)));
    SPIN_CUDA(cudaMalloc(&d->d_Mhat, ncplx * sizeof(cufftDoubleComplex)));
    SPIN_CUDA(cudaMalloc(&d->d_Hhat, ncplx * sizeof(cufftDoubleComplex)));
    SPIN_CUDA(cudaMalloc(&d->d_Khat, (size_t)nb * nb * 6 * d->Phalf * sizeof(cufftDoubleComplex)));
    SPIN_CUDA(cudaMalloc(&d->d_geom, (size_t)nb * sizeof(double)));
    SPIN_CUDA(cudaMemsetAsync(d->d_Mpad, 0, nreal * sizeof(double), s->stream));
    SPIN_CUDA(cudaMemcpyAsync(d->d_geom, s->mu.data(), nb * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    cufftHandle plan6 = 0;
    if (want_slab) {
        int na[1] = {d->P[0]}, nb1[1] = {d->P[1]};
        const int rows = s->nc[1] * d->SL, cols = d->SL * d->S1p;      // the pad columns of a row hold zeros and stay zero
        if (!d->own_a) {
            SPIN_FFT(cufftPlanMany(&d->plan_a_fwd, 1, na, na, 1, d->P[0], na, 1, d->S1p, CUFFT_D2Z, rows));
            SPIN_FFT(cufftPlanMany(&d->plan_a_inv, 1, na, na, 1, d->S1p, na, 1, d->P[0], CUFFT_Z2D, rows));
            SPIN_FFT(cufftSetStream(d->plan_a_fwd, s->stream));
            SPIN_FFT(cufftSetStream(d->plan_a_inv, s->stream));
        }
        if (!d->fused_b) {
            SPIN_FFT(cufftPlanMany(&d->plan_b, 1, nb1, nb1, cols, 1, nb1, cols, 1, CUFFT_Z2Z, cols));
            SPIN_FFT(cufftSetStream(d->plan_b, s->stream));
        }
        d->slab = true;      // from here on ddi_release destroys these plans
        // the twiddle table of every padded length (the same values whichever system uploads them)
        static double twr[17][16], twi[17][16];
        for (int pz = 1; pz <= 16; ++pz)
            for (int t = 0; t < 16; ++t) {
                twr[pz][t] = cos(-2.0 * M_PI * t / pz); twi[pz][t] = sin(-2.0 * M_PI * t / pz);
                if ((4 * t) % pz == 0) { const int k = ((4 * t) / pz) % 4; twr[pz][t] = k == 0 ? 1 : k == 2 ? -1 : 0; twi[pz][t] = k == 1 ? -1 : k == 3 ? 1 : 0; }   // exact at quarter turns
            }
        SPIN_CUDA(cudaMemcpyToSymbolAsync(DDI_TWR, twr, sizeof(twr), 0, cudaMemcpyHostToDevice, s->stream));
        SPIN_CUDA(cudaMemcpyToSymbolAsync(DDI_TWI, twi, sizeof(twi), 0, cudaMemcpyHostToDevice, s->stream));
        if (d->own_a) {
            // exp(-2 pi i t / P), t < P, exact at the multiples of an eighth of a turn
            auto upload_table = [&](const int P, double2 **dst) -> int {
                std::vector<double2> tw((size_t)P);
                for (int t = 0; t < P; ++t) {
                    tw[(size_t)t] = make_double2(cos(-2.0 * M_PI * t / P), sin(-2.0 * M_PI * t / P));
                    if ((8 * t) % P == 0) {
                        const int k = (8 * t) / P;
                        const double h = 0.70710678118654752440;
                        const double cr[8] = {1, h, 0, -h, -1, -h, 0, h}, ci[8] = {0, -h, -1, -h, 0, h, 1, h};
                        tw[(size_t)t] = make_double2(cr[k], ci[k]);
                    }
                }
                SPIN_CUDA(cudaMalloc(dst, (size_t)P * sizeof(double2)));
                SPIN_CUDA(cudaMemcpyAsync(*dst, tw.data(), (size_t)P * sizeof(double2), cudaMemcpyHostToDevice, s->stream));
                SPIN_CUDA(cudaStreamSynchronize(s->stream));      // tw is a local
                return SPIN_OK;
            };
            if (int rc = upload_table(d->P[0], &d->d_tw)) return rc;
            const int M = d->P[0] / 2;
            d->a_rows_per_block = M <= 256 ? 8 : (M <= 512 ? 4 : (M <= 1024 ? 2 : 1));
            d->a_smem = (size_t)d->a_rows_per_block * (2 * (M + M / 8) + 1) * sizeof(double2);
            SPIN_CUDA(cudaFuncSetAttribute(ddi_apass_fwd_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->a_smem));
            SPIN_CUDA(cudaFuncSetAttribute(ddi_apass_inv_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->a_smem));
            SPIN_CUDA(cudaFuncSetAttribute(ddi_apass_fwd_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->a_smem));
            SPIN_CUDA(cudaFuncSetAttribute(ddi_apass_inv_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->a_smem));
            if (d->fused_b) if (int rc = upload_table(d->P[1], &d->d_tw_b)) return rc;
            d->a256 = d->fused_b && M == 256 && Nb_ % DDI_A256_ROWS == 0;
            d->b256 = d->fused_b && Nb_ == 256;
            if (d->a256) {
                SPIN_CUDA(cudaFuncSetAttribute(ddi_apass256_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DDI_A256_SMEM));
                SPIN_CUDA(cudaFuncSetAttribute(ddi_apass256_inv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DDI_A256_SMEM));
            }
        }
    }
    if (d->rank > 0) {
        if (!want_slab) {
            SPIN_FFT(cufftPlanMany(&d->plan_r2c, d->rank, d->fdims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, nb * 3));
            SPIN_FFT(cufftPlanMany(&d->plan_c2r, d->rank, d->fdims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_Z2D, nb * 3));
            d->have_plans = true;
            SPIN_FFT(cufftSetStream(d->plan_r2c, s->stream));
            SPIN_FFT(cufftSetStream(d->plan_c2r, s->stream));
        }
        SPIN_FFT(cufftPlanMany(&plan6, d->rank, d->fdims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, 6));
        SPIN_FFT(cufftSetStream(plan6, s->stream));
    }
    // dipole tensor per sublattice pair: real-space image sums, then one batched transform of the 6 components
    DdiGeom G;
    for (int k = 0; k < 9; ++k) G.brav[k] = s->brav[k] * s->alat;
    for (int k = 0; k < 3 * nb; ++k) G.basis[k] = s->basis[k];
    for (int k = 0; k < 3; ++k) { G.N[k] = s->nc[k]; G.P[k] = d->P[k]; G.img[k] = s->per[k] ? s->ddi_img[k] : 0; }
    double *d_K6 = nullptr;
    SPIN_CUDA(cudaMalloc(&d_K6, (size_t)6 * d->Ptot * sizeof(double)));
    const int nt = 128;
    const unsigned nblk = (unsigned)((d->Ptot + nt - 1) / nt);
    for (int a = 0; a < nb; ++a)
        for (int b = 0; b < nb; ++b) {
            ddi_tensor_kernel<<<nblk, nt, 0, s->stream>>>(G, a, b, (long long)d->Ptot, d_K6);
            s->n_launch++;
            cufftDoubleComplex *dst = d->d_Khat + (size_t)(a * nb + b) * 6 * d->Phalf;
            if (d->rank > 0) { SPIN_FFT(cufftExecD2Z(plan6, d_K6, dst)); s->n_fft++; }
            else { real_to_complex_kernel<<<1, 32, 0, s->stream>>>(d_K6, dst, 6); s->n_launch++; }
        }
    if (want_slab && nb == 1) {       // keep the real part only (exactly real for one basis atom: K(-Delta) = K(Delta))
        const long long nk = (long long)6 * d->Phalf;
        SPIN_CUDA(cudaMalloc(&d->d_Kre, (size_t)nk * sizeof(double)));
        real_part_kernel<<<(unsigned)((nk + 255) / 256), 256, 0, s->stream>>>(d->d_Khat, d->d_Kre, nk);
        s->n_launch++;
        // mirror symmetry along c, checked on the numbers themselves (relative 1e-13; rounding of the transform leaves about 1e-16)
        unsigned long long *d_chk = nullptr, h_chk[2] = {0ull, 0ull};
        SPIN_CUDA(cudaMalloc(&d_chk, 2 * sizeof(unsigned long long)));
        SPIN_CUDA(cudaMemsetAsync(d_chk, 0, 2 * sizeof(unsigned long long), s->stream));
        ddi_mirror_check_kernel<<<(unsigned)((nk + 255) / 256), 256, 0, s->stream>>>(d->d_Kre, d->PZ, (long long)d->S2, d_chk);
        s->n_launch++;
        SPIN_CUDA(cudaMemcpyAsync(h_chk, d_chk, sizeof(h_chk), cudaMemcpyDeviceToHost, s->stream));
        SPIN_CUDA(cudaStreamSynchronize(s->stream));
        cudaFree(d_chk);
        double dev, mag;
        memcpy(&dev, &h_chk[0], 8); memcpy(&mag, &h_chk[1], 8);
        d->mirror = d->PZ > 2 && dev <= 1e-13 * mag && s->opt_ddi_mirror;
        if (d->fused_b) {      // the tensor in the fused kernel's order; the [6][PZ][S2] copy is not needed any more
            const int Mb = s->nc[1], NPL = d->mirror ? d->PZ / 2 + 1 : d->PZ;
            const long long nkb = (long long)d->S1 * 2 * 6 * NPL * Mb;
            SPIN_CUDA(cudaMalloc(&d->d_Kb, (size_t)nkb * sizeof(double)));
            ddi_bfused_tensor_kernel<<<(unsigned)((nkb + 255) / 256), 256, 0, s->stream>>>(d->d_Kre, d->d_Kb, d->PZ, NPL, Mb, d->S1);
            s->n_launch++;
            SPIN_CUDA(cudaStreamSynchronize(s->stream));
            cudaFree(d->d_Kre); d->d_Kre = nullptr;
#define SPIN_BF_ATTR(NZ_) case NZ_: \
            SPIN_CUDA(cudaFuncSetAttribute(ddi_bfused_kernel<NZ_, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->bf_smem)); \
            SPIN_CUDA(cudaFuncSetAttribute(ddi_bfused_kernel<NZ_, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->bf_smem)); \
            SPIN_CUDA(cudaFuncSetAttribute(ddi_bfused_kernel<NZ_, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->bf_smem)); \
            SPIN_CUDA(cudaFuncSetAttribute(ddi_bfused_kernel<NZ_, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->bf_smem)); break
            if (d->PZ == 1) {      // a monolayer, not padded along c
                SPIN_CUDA(cudaFuncSetAttribute(ddi_bfused_kernel<1, false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->bf_smem));
                SPIN_CUDA(cudaFuncSetAttribute(ddi_bfused_kernel<1, false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)d->bf_smem));
            } else switch (d->NZ) {
                SPIN_BF_ATTR(1); SPIN_BF_ATTR(2); SPIN_BF_ATTR(3); SPIN_BF_ATTR(4); SPIN_BF_ATTR(5); SPIN_BF_ATTR(6); SPIN_BF_ATTR(7); SPIN_BF_ATTR(8);
                default: return spin::fail(SPIN_ERR_STATE, "dipolar slab path: %d planes not supported", d->NZ);
            }
#undef SPIN_BF_ATTR
        }
    }
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    SPIN_CUDA(cudaGetLastError());
    cudaFree(d_K6);
    if (plan6) cufftDestroy(plan6);
    if (want_slab && nb == 1) { cudaFree(d->d_Khat); d->d_Khat = nullptr; }
    return SPIN_OK;
}

int spin::ddi_field(spin_system *s, const double *d_n, double *d_f) {
    DdiState *d = s->ddi;
    if (!d) return spin::fail(SPIN_ERR_STATE, "dipolar plan missing");
    const int nb = s->nb, Ncell = (int)s->ncell, nspin = nb * Ncell, nt = 256;
    const unsigned gs = (unsigned)((nspin + nt - 1) / nt);
    if (d->slab) {
        const int a_rows = s->nc[1] * d->SL;
        const unsigned ga = d->own_a ? (unsigned)((a_rows + d->a_rows_per_block - 1) / d->a_rows_per_block) : 0u;
        if (d->fused_b) {      // a-pass into [ka][slab][ib]; b-pass, c-pass, contraction and their inverses in one kernel; inverse a-pass
            const int Ma = d->P[0] / 2, Mb = s->nc[1];
            const size_t part1 = (size_t)d->S1 * d->SL * Mb;
            int lgMb = 0;
            while ((1 << lgMb) < Mb) ++lgMb;
            if (d->a256)
                SPIN_CUDA(ddi_launch(s, ddi_apass256_fwd_kernel, a_rows / DDI_A256_ROWS, 256, DDI_A256_SMEM, s->plan, d_n, d->SL, (const double *)d->d_geom,
                                     (const double2 *)d->d_tw, d->s_a));
            else
                SPIN_CUDA(ddi_launch(s, ddi_apass_fwd_kernel<true>, ga, 32 * d->a_rows_per_block, d->a_smem, s->plan, d_n, Ma, d->SL, d->S1p, a_rows,
                                     d->a_rows_per_block, (const double *)d->d_geom, (const double2 *)d->d_tw, d->s_a));
            if (s->profile_on) cudaEventRecord(s->ev2, s->stream);
#define SPIN_BF1(NZ_, MIR_, ...) SPIN_CUDA(ddi_launch(s, ddi_bfused_kernel<NZ_, MIR_, __VA_ARGS__>, 2 * d->S1, DDI_BF_THREADS, d->bf_smem, (const double *)d->d_Kb, (const double2 *)d->s_a, \
                                                     (double2 *)d->s_d, lgMb, d->S1, (const double2 *)d->d_tw_b))
#define SPIN_BF(NZ_) case NZ_: \
            if (d->b256) { if (d->mirror) SPIN_BF1(NZ_, true, true); else SPIN_BF1(NZ_, false, true); } \
            else { if (d->mirror) SPIN_BF1(NZ_, true, false); else SPIN_BF1(NZ_, false, false); } break
            if (d->PZ == 1) { if (d->b256) SPIN_BF1(1, false, true, false); else SPIN_BF1(1, false, false, false); }
            else switch (d->NZ) {
                SPIN_BF(1); SPIN_BF(2); SPIN_BF(3); SPIN_BF(4); SPIN_BF(5); SPIN_BF(6); SPIN_BF(7); SPIN_BF(8);
                default: return spin::fail(SPIN_ERR_STATE, "dipolar slab path: %d planes not supported", d->NZ);
            }
#undef SPIN_BF
#undef SPIN_BF1
            if (s->profile_on) {      // the fused kernel alone (bench.py's roofline kernel on dipolar workloads)
                cudaEventRecord(s->ev3, s->stream); cudaEventSynchronize(s->ev3);
                float ms = 0.f; cudaEventElapsedTime(&ms, s->ev2, s->ev3);
                s->prof_ms[3] += ms; s->prof_n[3]++;
            }
            if (d->a256)
                SPIN_CUDA(ddi_launch(s, ddi_apass256_inv_kernel, a_rows / DDI_A256_ROWS, 256, DDI_A256_SMEM, s->plan, (const cufftDoubleComplex *)d->s_d, d->SL,
                                     (const double *)d->d_geom, C_DD / (double)d->Ptot, (const double2 *)d->d_tw, d_f, part1));
            else
                SPIN_CUDA(ddi_launch(s, ddi_apass_inv_kernel<true>, ga, 32 * d->a_rows_per_block, d->a_smem, s->plan, (const cufftDoubleComplex *)d->s_d, Ma, d->SL,
                                     d->S1p, a_rows, d->a_rows_per_block, (const double *)d->d_geom, C_DD / (double)d->Ptot, (const double2 *)d->d_tw, d_f, part1));
            s->n_launch += 3;
            return SPIN_OK;
        }
        if (d->own_a) {                                                               // scatter + a-pass over the occupied rows, one kernel
            ddi_apass_fwd_kernel<false><<<ga, 32 * d->a_rows_per_block, d->a_smem, s->stream>>>(s->plan, d_n, d->P[0] / 2, d->SL, d->S1p, a_rows, d->a_rows_per_block,
                                                                                        d->d_geom, d->d_tw, d->s_a);
        } else {
            ddi_slab_scatter_kernel<<<gs, nt, 0, s->stream>>>(s->plan, d_n, d->P[0], d->SL, d->d_geom, d->s_in);
            SPIN_FFT(cufftExecD2Z(d->plan_a_fwd, d->s_in, d->s_a));                   // a-pass over the occupied rows only
        }
        SPIN_FFT(cufftExecZ2Z(d->plan_b, d->s_a, d->s_b, CUFFT_FORWARD));            // b-pass
        const unsigned gq = (unsigned)((d->S2 + DDI_CT_COLS - 1) / DDI_CT_COLS);
#define SPIN_CONTRACT(NZ_, PAD_, MIR_) ddi_slab_contract_kernel<NZ_, PAD_, MIR_><<<gq, 2 * DDI_CT_COLS, 0, s->stream>>>(d->d_Kre, d->s_b, d->s_b, (long long)d->S2, d->S1, d->S1p)
#define SPIN_CONTRACT_NZ(NZ_) case NZ_: if (d->mirror) SPIN_CONTRACT(NZ_, true, true); else SPIN_CONTRACT(NZ_, true, false); break
        if (s->profile_on) cudaEventRecord(s->ev2, s->stream);
        cufftDoubleComplex *spec_out = d->s_b;                                          // what the inverse b-pass reads
        if (nb > 1) {                                                                   // several sublattices: complex tensors, out of place
            const dim3 gm(gq, (unsigned)nb);
#define SPIN_CONTRACT_MB(NZ_, PAD_) ddi_slab_contract_mb_kernel<NZ_, PAD_><<<gm, 2 * DDI_CT_COLS, 0, s->stream>>>(d->d_Khat, d->s_b, d->s_c, nb, (long long)d->S2, d->S1, d->S1p)
            if (d->PZ == 1) SPIN_CONTRACT_MB(1, false);
            else switch (d->NZ) {
                case 1: SPIN_CONTRACT_MB(1, true); break;
                case 2: SPIN_CONTRACT_MB(2, true); break;
                case 3: SPIN_CONTRACT_MB(3, true); break;
                case 4: SPIN_CONTRACT_MB(4, true); break;
                default: return spin::fail(SPIN_ERR_STATE, "dipolar slab path: %d planes with %d sublattices not supported", d->NZ, nb);
            }
#undef SPIN_CONTRACT_MB
            spec_out = d->s_c;
        } else if (d->PZ == 1) SPIN_CONTRACT(1, false, false);                          // a single unpadded plane: contraction only
        else switch (d->NZ) {                                                           // c-pass + contraction + inverse c-pass, in place
            SPIN_CONTRACT_NZ(1); SPIN_CONTRACT_NZ(2); SPIN_CONTRACT_NZ(3); SPIN_CONTRACT_NZ(4);
            SPIN_CONTRACT_NZ(5); SPIN_CONTRACT_NZ(6); SPIN_CONTRACT_NZ(7); SPIN_CONTRACT_NZ(8);
            default: return spin::fail(SPIN_ERR_STATE, "dipolar slab path: %d planes not supported", d->NZ);
        }
#undef SPIN_CONTRACT_NZ
#undef SPIN_CONTRACT
        if (s->profile_on) {      // the contraction alone (bench.py's roofline kernel on dipolar workloads)
            cudaEventRecord(s->ev3, s->stream); cudaEventSynchronize(s->ev3);
            float ms = 0.f; cudaEventElapsedTime(&ms, s->ev2, s->ev3);
            s->prof_ms[3] += ms; s->prof_n[3]++;
        }
        SPIN_FFT(cufftExecZ2Z(d->plan_b, spec_out, d->s_d, CUFFT_INVERSE));          // inverse b-pass
        if (d->own_a) {                                                               // inverse a-pass + gather, one kernel
            ddi_apass_inv_kernel<false><<<ga, 32 * d->a_rows_per_block, d->a_smem, s->stream>>>(s->plan, d->s_d, d->P[0] / 2, d->SL, d->S1p, a_rows, d->a_rows_per_block,
                                                                                        d->d_geom, C_DD / (double)d->Ptot, d->d_tw, d_f, 0);
            s->n_launch += 3; s->n_fft += 2;
        } else {
            SPIN_FFT(cufftExecZ2D(d->plan_a_inv, d->s_d, d->s_out));                  // inverse a-pass, occupied rows only
            ddi_slab_gather_kernel<<<gs, nt, 0, s->stream>>>(s->plan, d->s_out, d->P[0], d->SL, d->d_geom, C_DD / (double)d->Ptot, d_f);
            s->n_launch += 3; s->n_fft += 4;
        }
        return SPIN_OK;
    }
    ddi_scatter_kernel<<<gs, nt, 0, s->stream>>>(s->plan, d_n, d->P[0], d->P[1], (long long)d->Ptot, d->d_geom, d->d_Mpad);
    s->n_launch++;
    if (d->rank > 0) { SPIN_FFT(cufftExecD2Z(d->plan_r2c, d->d_Mpad, d->d_Mhat)); s->n_fft++; }
    else { real_to_complex_kernel<<<1, 32, 0, s->stream>>>(d->d_Mpad, d->d_Mhat, nb * 3); s->n_launch++; }
    dim3 gc((unsigned)((d->Phalf + nt - 1) / nt), nb);
    ddi_contract_kernel<<<gc, nt, 0, s->stream>>>(d->d_Khat, d->d_Mhat, d->d_Hhat, nb, (long long)d->Phalf);
    s->n_launch++;
    if (d->rank > 0) { SPIN_FFT(cufftExecZ2D(d->plan_c2r, d->d_Hhat, d->d_Hpad)); s->n_fft++; }
    else { complex_to_real_kernel<<<1, 32, 0, s->stream>>>(d->d_Hhat, d->d_Hpad, nb * 3); s->n_launch++; }
    ddi_gather_kernel<<<gs, nt, 0, s->stream>>>(s->plan, d->d_Hpad, d->P[0], d->P[1], (long long)d->Ptot, d->d_geom,
                                                 C_DD / (double)d->Ptot, d_f);
    s->n_launch++;
    return SPIN_OK;
}
