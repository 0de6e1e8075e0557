// spin_jit_march.cuh -- the whole Depondt step (B5-B7) of a 3-D lattice in ONE pass: a plane-marching kernel
// (sm_100a; included by spin_jit_kernels.cuh when SPIN_MARCH is defined; Depondt or Heun solver, no dipolar term; one basis atom by
// default, up to four on request; flat lattices are the special case of one plane).
//
// Why.  The two brick sweeps move 120 B per spin-update through HBM (n^p written and read back, n read twice), fetch every line
// 2.8 times from L2 (brick halos) and evaluate F(n) twice.  On B200 that is not bandwidth- but POWER-bound: a 2-s run of cfg3 sits at
// the 1000 W cap and the SM clock falls from 1965 to about 1650 MHz (profiles/r2_README.md).  This kernel removes the n^p round trip,
// the second evaluation of F(n) and most of the L2 re-fetches:
//   * a block owns a column of 32 x TY sites and marches along c through a chunk of planes;
//   * one elected thread streams the n planes (tile + a rim of twice the Hamiltonian's reach) into a shared-memory ring with one TMA
//     tensor copy per plane (cp.async.bulk.tensor, completion on an mbarrier), two planes ahead of the compute;
//   * per iteration every thread computes the PREDICTOR of one site of plane zP -- tile plus a rim of one reach: TY + 2 RB aligned rows of
//     32 sites by as many warps, the 2 RA rim columns by extra warps -- and writes n^p into a second ring that never leaves the SM;
//   * after one __syncthreads the tile's threads compute the CORRECTOR of plane zP - RC from that ring: A(n), n and the thermal field of
//     their site are still in their registers, so F(n) is evaluated once per step, and write n(t + dt) (and its periodic images).
// The arithmetic is the brick kernels' (force<>, rotation_field<>, rodrigues, same order): results are bit-identical (tested).
// Ghost layers are twice the reach wide in this mode (the planner doubles them): the rim predictor needs n two reaches out.
// HBM traffic: read n once (+ chunk overlap), write n once = 48-60 B per spin-update instead of 120.
//
// spec must also define: int MRA, MRB, MRC (reach of the Hamiltonian; ghost widths RA, RB, RC are twice that), MTY (rows per tile),
// MNZC (chunks along c), MLOOK (planes of look-ahead), MBLOCKS (blocks per SM the geometry was planned for).
#pragma once

namespace spinmarch {
using namespace spinjit;

struct __align__(64) TensorMap { unsigned long long opaque[16]; };      // CUtensorMap, passed as a __grid_constant__ parameter
template <int V> struct spin_ddi_like_int { static constexpr int value = V; };

constexpr int RA = spec::MRA, RB = spec::MRB, RC = spec::MRC, TY = spec::MTY, NZC = spec::MNZC;
constexpr int HX = (2 * RA + 1) / 2 * 2;                         // rim of a staged n row, even: TMA box rows start 16-byte aligned
constexpr int NX = 32 + 2 * HX, NY = TY + 4 * RB;                // staged n plane (rim of two reaches), sites
constexpr int NBS = spec::NBASIS;                                // sublattices: each has its own sub-slot in a staged plane
constexpr int NROW = 3 * NX, NPL = NROW * NY, NSLOTB = (NPL + 15) / 16 * 16, NSLOT = NBS * NSLOTB;      // doubles; (sub-)slots are 128-byte multiples
constexpr int PX = 32 + 2 * RA, PY = TY + 2 * RB;                // n^p plane (rim of one reach)
constexpr int PROW = 3 * PX, PPLB = PROW * PY, PPL = NBS * PPLB;
constexpr int LOOK = spec::MLOOK;                                // n planes in flight beyond the ones the current predictor reads
constexpr int RN = 2 * RC + 1 + LOOK, RP = 2 * RC + 2;           // ring depths: n planes, n^p planes
constexpr int RIM = 2 * RA * PY, RIMW = (RIM + 31) / 32;         // sites of the rim columns, warps that take them
constexpr int NWARP = PY + RIMW, NTHREADS = 32 * NWARP;
constexpr int NTX = (spec::NA + 31) / 32, NTY = (spec::NB + TY - 1) / TY;
static_assert(spec::NBASIS <= 4 && (spec::SOLVER == 0 || spec::SOLVER == 1) && !spec::HAS_DDI && !spec::MULTI_IMAGE, "one-pass kernel: up to four basis atoms, Depondt or Heun, no dipolar term");
// the TMA descriptors of the sublattices' arrays (same shape, different base)
struct __align__(64) TensorMaps { TensorMap m[NBS]; };
template <int B = 0, class F> __device__ __forceinline__ void for_each_basis(F &&f) {
    if constexpr (B < NBS) { f(spin_ddi_like_int<B>{}); for_each_basis<B + 1>(f); }
}
static_assert(spec::RA == 2 * RA && spec::RB == 2 * RB && spec::RC == 2 * RC, "ghost layers must be twice the reach");

extern __shared__ __align__(128) double smem[];

__device__ __forceinline__ u32 smem_u32(const void *p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u32 bar, u32 count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(u32 bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(u32 bar, u32 parity) {
    u32 done = 0;
    for (int spin = 0; !done; ++spin) {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (spin > (1 << 24)) __trap();      // a lost copy must end the launch with an error, never hang the device
    }
}
__device__ __forceinline__ void tma_load_4d(u32 dst, const TensorMap *tm, int c0, int c1, int c2, int c3, u32 bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}

// partner of a site in a ring of staged planes: pl[dz + RC] points at the x component of the own site in the plane z + dz
template <int XS, int ROWS, int SUBS>      // doubles between the components of a row (= sites per row), between rows, between sublattices
struct RingAcc {
    const double *pl[2 * RC + 1];            // (of the sublattice B the accessor was set up for)
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int, double (&v)[3]) const {
        const double *q = pl[DC + RC] + ((BJ - B) * SUBS + DB * ROWS + DA);
        v[0] = q[0]; v[1] = q[XS]; v[2] = q[2 * XS];
    }
};
}  // namespace spinmarch

extern "C" __global__ void __launch_bounds__(spinmarch::NTHREADS, spec::MBLOCKS)
    jit_depondt_march(const __grid_constant__ spinmarch::TensorMaps tm_n, double *__restrict__ nout, const unsigned long long *__restrict__ d_step,
                      unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi, const unsigned char *__restrict__ pin,
                      const double *__restrict__ mu_ratio, unsigned int item0, double *__restrict__ peer_lo, double *__restrict__ peer_hi,
                      int peer_lo_nc) {
    using namespace spinmarch;
    const unsigned long long step = *d_step + step_add;
    const int item = (int)(blockIdx.x + item0), col = item % (NTX * NTY), chunk = item / (NTX * NTY);      // (item0: a launch over a range of chunks)
    const int x0 = (col % NTX) * 32, y0 = (col / NTX) * TY;
    const int za = (int)((long long)chunk * spec::NC / NZC), zb = (int)((long long)(chunk + 1) * spec::NC / NZC);
    const int NP = zb - za + 4 * RC;                              // n planes za - 2 RC .. zb - 1 + 2 RC
    double *nring = smem, *pring = smem + RN * NSLOT;
    const u32 bars = smem_u32(pring + RP * PPL);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    auto issue = [&](int p) {
        const u32 bar = bars + 8u * (p % RN);
        mbar_expect_tx(bar, (u32)(NBS * NPL * 8));
#pragma unroll
        for (int b = 0; b < NBS; ++b)
            tma_load_4d(smem_u32(nring + (p % RN) * NSLOT + b * NSLOTB), &tm_n.m[b], spec::LA + x0 - HX, 0, spec::LB + y0 - 2 * RB, spec::LC + za - 2 * RC + p, bar);
    };
    if (tid == 0) {
        for (int s = 0; s < RN; ++s) mbar_init(bars + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) for (int p = 0; p < RN - 1 && p < NP; ++p) issue(p);
    // the site of this thread relative to the tile: the first PY warps hold the aligned rows, the others the rim columns
    int sx, sy;
    bool mine = true;
    if (warp < PY) { sx = lane; sy = warp - RB; }
    else {
        const int r = (warp - PY) * 32 + lane;                    // rim site: row r / (2 RA), column r % (2 RA)
        mine = r < RIM;
        const int cr = mine ? r % (2 * RA) : 0;
        sy = (mine ? r / (2 * RA) : 0) - RB;
        sx = cr < RA ? cr - RA : 32 + (cr - RA);
    }
    const int gx = x0 + sx, gy = y0 + sy;                          // lattice coordinates, possibly in the ghost region
    // a predictor site is live if it is a lattice site or the periodic image of one; elsewhere (open edges, tiles hanging over the
    // lattice) n^p is the zero vector, exactly what the ghost cells of the brick kernels hold there
    const bool live_xy = mine && (spec::PER_A ? (gx >= -RA && gx < spec::NA + RA) : (gx >= 0 && gx < spec::NA)) &&
                         (spec::PER_B ? (gy >= -RB && gy < spec::NB + RB) : (gy >= 0 && gy < spec::NB));
    const bool tile_site = warp < PY && sy >= 0 && sy < TY && gx < spec::NA && gy < spec::NB;      // corrector sites
    Coord c;                                                       // the lattice site this one is (an image of)
    c.ia = gx < 0 ? gx + spec::NA : (gx >= spec::NA ? gx - spec::NA : gx);
    c.ib = gy < 0 ? gy + spec::NB : (gy >= spec::NB ? gy - spec::NB : gy);
    const int ncell = ((sy + 2 * RB) * 3) * NX + (sx + HX);       // x component of the own site in a staged n plane
    const int pcell = ((sy + RB) * 3) * PX + (sx + RA);           // the same in an n^p plane
    // what the corrector of plane zC needs from the predictor of the same site, RC iterations earlier (flat lattices, RC = 0: the one
    // plane there is -- the predictor's values of this very iteration, and the queue is not used); one set per sublattice
    constexpr int QD = RC > 0 ? RC : 1;
    double n_q[QD][NBS][3], A_q[QD][NBS][3], th_q[QD][NBS][3];
#pragma unroll
    for (int r = 0; r < QD; ++r)
#pragma unroll
        for (int b = 0; b < NBS; ++b)
#pragma unroll
            for (int k = 0; k < 3; ++k) { n_q[r][b][k] = 0.0; A_q[r][b][k] = 0.0; th_q[r][b][k] = 0.0; }
#pragma unroll
    for (int p = 0; p < 2 * RC; ++p) mbar_wait(bars + 8u * p, 0u);
    const int NIT = zb - za + 2 * RC;
    // ring positions kept incrementally (no division in the loop): ns = k mod RN, ps = k mod RP, (wslot, wpar) = slot and parity of plane k + 2 RC
    int ns = 0, ps = 0, wslot = (2 * RC) % RN, wpar = ((2 * RC) / RN) & 1;
    auto nslot_of = [&](int d) { int t = ns + d; return t >= RN ? t - RN : t; };                 // slot of n plane k + d, 0 <= d <= 2 RC
    auto pslot_of = [&](int d) { int t = ps + d; return t < 0 ? t + RP : t; };                   // slot of n^p plane k + d, -2 RC <= d <= 0
    for (int k = 0; k < NIT; ++k) {                                // predictor plane zP = za - RC + k from n planes k .. k + 2 RC
        mbar_wait(bars + 8u * wslot, (u32)wpar);
        const int zP = za - RC + k;
        double n_cur[NBS][3], A_cur[NBS][3], th_cur[NBS][3];
#pragma unroll
        for (int b = 0; b < NBS; ++b)
#pragma unroll
            for (int q = 0; q < 3; ++q) { n_cur[b][q] = 0.0; A_cur[b][q] = 0.0; th_cur[b][q] = 0.0; }
        double *pslot = pring + ps * PPL;
        if (mine) {
            // plane of the WHOLE lattice (slab decomposition: planes beyond the slab are the neighbours', staged from the ghost layers the
            // halo exchange fills; their predictor is recomputed here like the rim of a tile)
            const int gz = spec::C_OFF + zP;
            const bool live = live_xy && (spec::PER_C || (gz >= 0 && gz < spec::GNC));
            if (live) c.ic = (gz < 0 ? gz + spec::GNC : (gz >= spec::GNC ? gz - spec::GNC : gz)) - spec::C_OFF;      // (outside [0, NC) only in a slab: noise index)
            for_each_basis([&](auto bc) {
                constexpr int B = decltype(bc)::value;
                double out[3] = {0.0, 0.0, 0.0};
                if (live) {
                    RingAcc<NX, NROW, NSLOTB> acc;
#pragma unroll
                    for (int dz = -RC; dz <= RC; ++dz) acc.pl[dz + RC] = nring + nslot_of(RC + dz) * NSLOT + B * NSLOTB + ncell;
                    double own[1][3], F[1][3], sg[1][3] = {{0.0, 0.0, 0.0}};
                    acc.template load<B, B, 0, 0, 0>(0, own[0]);
                    n_cur[B][0] = own[0][0]; n_cur[B][1] = own[0][1]; n_cur[B][2] = own[0][2];
                    if (is_pinned<B>(pin, c)) { out[0] = own[0][0]; out[1] = own[0][1]; out[2] = own[0][2]; }
                    else {
                        const double zr = site_ratio<B>(mu_ratio, c), ir = spec::HAS_SITE_MU ? 1.0 / zr : 1.0;      // per-site moment
                        const double sscale = (spec::HAS_SITE_MU && spec::THERMAL_ON) ? sqrt(zr) : 1.0;
                        thermal_force<B>(c, step, seed_lo, seed_hi, F[0], 0u, sscale);
                        th_cur[B][0] = F[0][0]; th_cur[B][1] = F[0][1]; th_cur[B][2] = F[0][2];
                        force<B, 1>(acc, own, F, zr);
                        if constexpr (spec::STT_ON) stt_gradient<B, 1>(acc, c, own, sg);
                        rotation_field<B>(own[0], F[0], sg[0], A_cur[B], ir);
                        if constexpr (spec::SOLVER == 1) { out[0] = own[0][0]; out[1] = own[0][1]; out[2] = own[0][2]; spin::heun_add(own[0], A_cur[B], specc::DT, out); }   // Heun, B3
                        else spin::rodrigues(A_cur[B], specc::DT, specc::DT2, own[0], out);          // Depondt, B5
                    }
                }
                double *pq = pslot + B * PPLB + pcell;
                pq[0] = out[0]; pq[PX] = out[1]; pq[2 * PX] = out[2];
            });
        }
        if constexpr (RC == 0) {
#pragma unroll
            for (int b = 0; b < NBS; ++b)
#pragma unroll
                for (int q = 0; q < 3; ++q) { n_q[0][b][q] = n_cur[b][q]; A_q[0][b][q] = A_cur[b][q]; th_q[0][b][q] = th_cur[b][q]; }
        }
        __syncthreads();                                           // n^p(zP) is complete; nobody reads n plane k any more
        if (tid == 0 && k + RN - 1 < NP) issue(k + RN - 1);        // refill a free slot, LOOK planes ahead of the next predictor
        const int zC = zP - RC;
        if (k >= 2 * RC && tile_site) {                            // corrector of plane zC from n^p planes zC - RC .. zC + RC = zP
            c.ic = zC;
            const size_t in_plane = (size_t)(c.ib + spec::LB) * ROW + (c.ia + spec::LA);
            for_each_basis([&](auto bc) {
                constexpr int B = decltype(bc)::value;
                double o[3];
                if (is_pinned<B>(pin, c)) { o[0] = n_q[0][B][0]; o[1] = n_q[0][B][1]; o[2] = n_q[0][B][2]; }
                else {
                    const double zr = site_ratio<B>(mu_ratio, c), ir = spec::HAS_SITE_MU ? 1.0 / zr : 1.0;
                    RingAcc<PX, PROW, PPLB> acc;
#pragma unroll
                    for (int dz = -RC; dz <= RC; ++dz) acc.pl[dz + RC] = pring + pslot_of(dz - RC) * PPL + B * PPLB + pcell;
                    double own[1][3], F[1][3] = {{th_q[0][B][0], th_q[0][B][1], th_q[0][B][2]}}, sg[1][3] = {{0.0, 0.0, 0.0}}, Ap[3];
                    acc.template load<B, B, 0, 0, 0>(0, own[0]);
                    force<B, 1>(acc, own, F, zr);
                    if constexpr (spec::STT_ON) stt_gradient<B, 1>(acc, c, own, sg);
                    rotation_field<B>(own[0], F[0], sg[0], Ap, ir);
                    if constexpr (spec::SOLVER == 1) {                                            // Heun, B4: n + dt/2 (n x A + n^p x A^p), renormalised
                        o[0] = n_q[0][B][0]; o[1] = n_q[0][B][1]; o[2] = n_q[0][B][2];
                        spin::heun_add(n_q[0][B], A_q[0][B], specc::HDT, o);
                        spin::heun_add(own[0], Ap, specc::HDT, o);
                        spin::renormalise_general(o);
                    } else {
                        const double Ac[3] = {A_q[0][B][0] + Ap[0], A_q[0][B][1] + Ap[1], A_q[0][B][2] + Ap[2]};
                        spin::rodrigues(Ac, specc::HDT, specc::QDT2, n_q[0][B], o);                // Depondt, B6-B7: R((A + A^p) / 2) n(t)
                        spin::renormalise(o);
                    }
                }
                const size_t site = (size_t)B * spec::SUB + in_plane;
                store_spin(nout + ((size_t)(zC + spec::LC) * PLANE + site), c, o);
                // Slab decomposition, fused exchange (llg_slab_step_fused): the planes a neighbouring slab holds as ghost layers are written
                // straight into ITS next configuration -- peer memory on another GPU (NVLink), or another array of this GPU -- with their
                // in-plane images; no halo copy follows.  peer_lo: the lower neighbour (its ghost layer above its peer_lo_nc planes),
                // peer_hi: the upper neighbour (its ghost layer below plane 0).  Same layout on every slab but for the number of planes.
                if constexpr (spec::SLAB && NBS == 1) {
                    if (peer_lo && zC < spec::LC) store_spin(peer_lo + ((size_t)(spec::LC + peer_lo_nc + zC) * PLANE + site), c, o);
                    if (peer_hi && zC >= spec::NC - spec::LC) store_spin(peer_hi + ((size_t)(zC - (spec::NC - spec::LC)) * PLANE + site), c, o);
                }
            });
        }
        // the queue moves on: slot 0 is the oldest (the plane the next corrector takes)
        if constexpr (RC > 0) {
#pragma unroll
            for (int b = 0; b < NBS; ++b) {
#pragma unroll
                for (int r = 0; r + 1 < RC; ++r)
#pragma unroll
                    for (int q = 0; q < 3; ++q) { n_q[r][b][q] = n_q[r + 1][b][q]; A_q[r][b][q] = A_q[r + 1][b][q]; th_q[r][b][q] = th_q[r + 1][b][q]; }
#pragma unroll
                for (int q = 0; q < 3; ++q) { n_q[QD - 1][b][q] = n_cur[b][q]; A_q[QD - 1][b][q] = A_cur[b][q]; th_q[QD - 1][b][q] = th_cur[b][q]; }
            }
        }
        if (++ns == RN) ns = 0;
        if (++ps == RP) ps = 0;
        if (++wslot == RN) { wslot = 0; wpar ^= 1; }
    }
}
