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
};

namespace {

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
__global__ void ddi_scatter_kernel(const __grid_constant__ DevicePlan L, const double *__restrict__ n, int P0, int P1, long long Ptot,
                                   const double *__restrict__ mu, double *__restrict__ Mpad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // b*Ncell + cell, x fastest
    if (i >= L.nb * L.Ncell) return;
    const int b = i / L.Ncell, cell = i - b * L.Ncell;
    const int ia = cell % L.Na, ib = (cell / L.Na) % L.Nb, ic = cell / (L.Na * L.Nb);
    const long long p = ia + (long long)P0 * (ib + (long long)P1 * ic);
    const int j = b * L.sub + ((ic + L.LC) * L.PB + (ib + L.LB)) * (3 * L.PA) + (ia + L.LA);
    const double m = mu[b];
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
    const double m = mu[b] * scale;
#pragma unroll
    for (int k = 0; k < 3; ++k) f[j + k * L.PA] = m * Hpad[(size_t)(b * 3 + k) * Ptot + p];
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

#define SPIN_FFT(call)                                                                                         \
    do {                                                                                                       \
        cufftResult r__ = (call);                                                                              \
        if (r__ != CUFFT_SUCCESS) return spin::fail(SPIN_ERR_CUDA, "%s failed: cufft error %d (%s:%d)", #call, \
                                                    (int)r__, __FILE__, __LINE__);                             \
    } while (0)

}  // namespace

void spin::ddi_release(spin_system *s) {
    DdiState *d = s->ddi;
    if (!d) return;
    if (d->have_plans) { cufftDestroy(d->plan_r2c); cufftDestroy(d->plan_c2r); }
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
    const size_t nreal = (size_t)nb * 3 * d->Ptot, ncplx = (size_t)nb * 3 * d->Phalf;
    SPIN_CUDA(cudaMalloc(&d->d_Mpad, nreal * sizeof(double)));
    SPIN_CUDA(cudaMalloc(&d->d_Hpad, nreal * sizeof(double)));
    SPIN_CUDA(cudaMalloc(&d->d_Mhat, ncplx * sizeof(cufftDoubleComplex)));
    SPIN_CUDA(cudaMalloc(&d->d_Hhat, ncplx * sizeof(cufftDoubleComplex)));
    SPIN_CUDA(cudaMalloc(&d->d_Khat, (size_t)nb * nb * 6 * d->Phalf * sizeof(cufftDoubleComplex)));
    SPIN_CUDA(cudaMalloc(&d->d_geom, (size_t)nb * sizeof(double)));
    SPIN_CUDA(cudaMemsetAsync(d->d_Mpad, 0, nreal * sizeof(double), s->stream));
    SPIN_CUDA(cudaMemcpyAsync(d->d_geom, s->mu.data(), nb * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    cufftHandle plan6 = 0;
    if (d->rank > 0) {
        SPIN_FFT(cufftPlanMany(&d->plan_r2c, d->rank, d->fdims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, nb * 3));
        SPIN_FFT(cufftPlanMany(&d->plan_c2r, d->rank, d->fdims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_Z2D, nb * 3));
        d->have_plans = true;
        SPIN_FFT(cufftSetStream(d->plan_r2c, s->stream));
        SPIN_FFT(cufftSetStream(d->plan_c2r, s->stream));
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
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    SPIN_CUDA(cudaGetLastError());
    cudaFree(d_K6);
    if (plan6) cufftDestroy(plan6);
    return SPIN_OK;
}

int spin::ddi_field(spin_system *s, const double *d_n, double *d_f) {
    DdiState *d = s->ddi;
    if (!d) return spin::fail(SPIN_ERR_STATE, "dipolar plan missing");
    const int nb = s->nb, Ncell = (int)s->ncell, nspin = nb * Ncell, nt = 256;
    const unsigned gs = (unsigned)((nspin + nt - 1) / nt);
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
