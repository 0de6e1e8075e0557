// spin_device_math.cuh -- device-only arithmetic shared by the table-driven kernels (spin_kernels.cuh) and the
// run-time specialised kernels (spin_jit_kernels.cuh).  No host headers: this file is also compiled by NVRTC.
//
//   thermal noise   Eq. 11: three standard normals per spin and step from Philox4x32-10
//   R(A) n          App. B: rotation that integrates dn/dt = n x A exactly for constant A
#pragma once

namespace spin {

// ---------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011) and the thermal triple (R13): key = seed, counter =
// (spin, block, step_lo, step_hi); uniforms from the top 53 of 64 bits (+1/2 ulp); Box-Muller.
__device__ __forceinline__ void philox4x32_10(unsigned int &c0, unsigned int &c1, unsigned int &c2, unsigned int &c3, unsigned int k0, unsigned int k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned int h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const unsigned int h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        const unsigned int n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}
__device__ __forceinline__ double uniform53(unsigned int hi, unsigned int lo) {
    const unsigned long long v = (((unsigned long long)hi << 32) | lo) >> 11;
    return ((double)v + 0.5) * (1.0 / 9007199254740992.0);
}
// image m of a batched system draws from the counter words block + 2 m (R30); image 0 is the single-system stream
__device__ __forceinline__ void thermal_xi(unsigned int seed_lo, unsigned int seed_hi, unsigned long long step, unsigned int spin, double (&xi)[3],
                                           unsigned int image = 0u) {
    unsigned int a0 = spin, a1 = 2u * image, a2 = (unsigned int)step, a3 = (unsigned int)(step >> 32);
    philox4x32_10(a0, a1, a2, a3, seed_lo, seed_hi);
    double sn, cs;
    double rad = sqrt(-2.0 * log(uniform53(a0, a1)));
    sincospi(2.0 * uniform53(a2, a3), &sn, &cs);
    xi[0] = rad * cs;
    xi[1] = rad * sn;
    unsigned int b0 = spin, b1 = 2u * image + 1u, b2 = (unsigned int)step, b3 = (unsigned int)(step >> 32);
    philox4x32_10(b0, b1, b2, b3, seed_lo, seed_hi);
    rad = sqrt(-2.0 * log(uniform53(b0, b1)));
    xi[2] = rad * cospi(2.0 * uniform53(b2, b3));
}

// R(A) n: Rodrigues rotation about -A/|A| by theta = |A| dt (exact flow of dn/dt = n x A for constant A).
// Written without square root or division:  with x = theta^2,
//     n' = n (1 - x q(x)) - (A x n) dt s(x) + A (A.n) dt^2 q(x),   s = sin(theta)/theta,  q = (1 - cos(theta))/theta^2
// s and q are even power series in theta: s = sum_k ROD_S[k] x^k, q = sum_k ROD_Q[k] x^k.  For x < 2^-10 (theta < 0.031 rad,
// every step of the paper's workloads) degree 4 is exact to 2e-23; for x < 1/4 degree 8 to 1e-18; larger angles take the
// trigonometric branch.  The coefficients live in constant memory: an fp64 operand from the constant bank costs no
// instruction, a 64-bit immediate costs two moves.
__constant__ double ROD_S[9] = {1.0, -1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0, 1.0 / 6227020800.0,
                                -1.0 / 1307674368000.0, 1.0 / 355687428096000.0};                       // (-1)^k / (2k+1)!
__constant__ double ROD_Q[9] = {0.5, -1.0 / 24.0, 1.0 / 720.0, -1.0 / 40320.0, 1.0 / 3628800.0, -1.0 / 479001600.0, 1.0 / 87178291200.0,
                                -1.0 / 20922789888000.0, 1.0 / 6402373705728000.0};                     // (-1)^k / (2k+2)!
__device__ __forceinline__ void rodrigues(const double (&A)[3], double dt, double dt2, const double (&n)[3], double (&out)[3]) {
    // every product and sum below is written out (fma / __dmul_rn): the compiler has no freedom to contract differently in different
    // kernels, so all sweep variants give the same bits
    const double a2 = fma(A[0], A[0], fma(A[1], A[1], __dmul_rn(A[2], A[2])));
    const double x = __dmul_rn(a2, dt2);
    double s, q;
    if (x < 0x1p-10) {
        s = fma(fma(fma(fma(ROD_S[4], x, ROD_S[3]), x, ROD_S[2]), x, ROD_S[1]), x, ROD_S[0]);
        q = fma(fma(fma(fma(ROD_Q[4], x, ROD_Q[3]), x, ROD_Q[2]), x, ROD_Q[1]), x, ROD_Q[0]);
    } else if (x < 0.25) {
        s = ROD_S[8]; q = ROD_Q[8];
#pragma unroll
        for (int k = 7; k >= 0; --k) { s = fma(s, x, ROD_S[k]); q = fma(q, x, ROD_Q[k]); }
    } else {
        const double th = sqrt(x);
        double sn, cs;
        sincos(th, &sn, &cs);
        s = sn / th;
        q = (1.0 - cs) / x;
    }
    const double c = fma(-x, q, 1.0);
    const double ds = __dmul_rn(dt, s);
    const double an = __dmul_rn(__dmul_rn(fma(A[0], n[0], fma(A[1], n[1], __dmul_rn(A[2], n[2]))), dt2), q);
    const double cx = fma(A[1], n[2], -__dmul_rn(A[2], n[1])), cy = fma(A[2], n[0], -__dmul_rn(A[0], n[2])), cz = fma(A[0], n[1], -__dmul_rn(A[1], n[0]));
    out[0] = fma(A[0], an, fma(-cx, ds, __dmul_rn(n[0], c)));
    out[1] = fma(A[1], an, fma(-cy, ds, __dmul_rn(n[1], c)));
    out[2] = fma(A[2], an, fma(-cz, ds, __dmul_rn(n[2], c)));
}

// Implicit-midpoint structure of the SIB solver (App. C, C5-C10): x + A' x x = n + n x A' with A' = (dt/2) A.
// The paper solves the 3x3 system by Cramer's rule; its closed form is x = [a + A'(a.A') - A' x a] / (1 + |A'|^2), a = n + n x A'
// (dot the equation with A' for x.A' = a.A', cross it with A' and eliminate A' x x).  |x| = |n| exactly (Cayley transform).
__device__ __forceinline__ void imp_update(const double (&A)[3], double hdt, const double (&n)[3], double (&out)[3]) {
    const double Ah[3] = {__dmul_rn(hdt, A[0]), __dmul_rn(hdt, A[1]), __dmul_rn(hdt, A[2])};
    const double a[3] = {n[0] + fma(n[1], Ah[2], -__dmul_rn(n[2], Ah[1])), n[1] + fma(n[2], Ah[0], -__dmul_rn(n[0], Ah[2])),
                         n[2] + fma(n[0], Ah[1], -__dmul_rn(n[1], Ah[0]))};
    const double aA = fma(a[0], Ah[0], fma(a[1], Ah[1], __dmul_rn(a[2], Ah[2])));
    const double inv = 1.0 / (1.0 + fma(Ah[0], Ah[0], fma(Ah[1], Ah[1], __dmul_rn(Ah[2], Ah[2]))));
    out[0] = __dmul_rn(fma(Ah[0], aA, a[0]) - fma(Ah[1], a[2], -__dmul_rn(Ah[2], a[1])), inv);
    out[1] = __dmul_rn(fma(Ah[1], aA, a[1]) - fma(Ah[2], a[0], -__dmul_rn(Ah[0], a[2])), inv);
    out[2] = __dmul_rn(fma(Ah[2], aA, a[2]) - fma(Ah[0], a[1], -__dmul_rn(Ah[1], a[0])), inv);
}

// Heun (App. B, B3-B4) with f = n x A:  f(n, A) added to `acc` with weight w
__device__ __forceinline__ void heun_add(const double (&n)[3], const double (&A)[3], double w, double (&acc)[3]) {
    acc[0] = fma(w, fma(n[1], A[2], -__dmul_rn(n[2], A[1])), acc[0]);
    acc[1] = fma(w, fma(n[2], A[0], -__dmul_rn(n[0], A[2])), acc[1]);
    acc[2] = fma(w, fma(n[0], A[1], -__dmul_rn(n[1], A[0])), acc[2]);
}

__device__ __forceinline__ void renormalise_general(double (&v)[3]) {      // Heun: |v| is not close to 1 to rounding
    const double sc = 1.0 / sqrt(fma(v[0], v[0], fma(v[1], v[1], __dmul_rn(v[2], v[2]))));
    v[0] *= sc; v[1] *= sc; v[2] *= sc;
}

__device__ __forceinline__ void renormalise(double (&v)[3]) {
    // |v|^2 = 1 + eps with eps ~ 1e-16 after a rotation of a unit vector: 1/sqrt(1+eps) by its series
    const double eps = fma(v[0], v[0], fma(v[1], v[1], fma(v[2], v[2], -1.0)));
    double sc;
    if (fabs(eps) < 1e-5) sc = fma(eps, fma(eps, fma(eps, -0.3125, 0.375), -0.5), 1.0);
    else sc = 1.0 / sqrt(1.0 + eps);
    v[0] *= sc; v[1] *= sc; v[2] *= sc;
}

}  // namespace spin
