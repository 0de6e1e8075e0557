// spin_jit_tma.cuh -- the two Depondt sweeps as persistent, TMA-fed plane-marching kernels (sm_100a; included by
// spin_jit_kernels.cuh when SPIN_TMA is defined).
//
// Why: the brick kernels (jit_predictor / jit_corrector) fetch every partner through L1 and wait for ~21 (42) loads before
// they compute; ncu shows them latency bound with L1/TEX at 75 %, L2 -> SM traffic at 2.5x the tile bytes, HBM at 41-48 %.
// Here the lattice is cut into columns of TBX x TBY cells; a CTA (one thread per cell of the column cross-section) marches
// along c through a chunk of CZ planes.  One elected thread streams whole planes (tile + ghost rim, all sublattices, x/y/z)
// into a ring of RING shared-memory slots with one 5-D TMA tensor copy per plane and array (cp.async.bulk.tensor, completion
// on an mbarrier), LOOK planes ahead of the compute.  Every partner read is then a shared-memory load at `slot[dz] + immediate`;
// each global line is fetched from L2 once per column (rim overhead (TBX+2r)(TBY+2r)/(TBX TBY), plus 2r planes per chunk).
// Results are written straight to global memory (coalesced rows, periodic images included, as in the brick kernels).
// The arithmetic is the same code as the brick kernels (force<>, rotation_field<>, rodrigues): only the accessor differs.
//
// spec must also define: struct TmaP, struct TmaC, each with static constexpr int TBX, TBY, KZ, RING, LOOK, NZC, CZ.
#pragma once

namespace spintma {
using namespace spinjit;

struct __align__(64) TensorMap { unsigned long long opaque[16]; };      // CUtensorMap, passed as a __grid_constant__ parameter

// geometry of one sweep's staging; G (spec::TmaP for the predictor, spec::TmaC for the corrector) gives TBX, TBY, RING, LOOK, NZC, CZ
template <class G>
struct Geo {
    static constexpr int TBX = G::TBX, TBY = G::TBY, RING = G::RING, LOOK = G::LOOK, NZC = G::NZC, CZ = G::CZ, KZ = G::KZ;
    static constexpr int HX = (spec::RA + 1) / 2 * 2;                     // rim along a, even: TMA needs 16-byte aligned box rows in global memory
    static constexpr int WX = TBX + 2 * HX, WY = TBY + 2 * spec::RB;      // staged box: cells incl. the ghost rim
    static constexpr int SROW = 3 * WX;                                   // doubles between rows of a staged plane (x, y, z runs)
    static constexpr int SSUB = SROW * WY;                                // doubles per sublattice of a staged plane
    static constexpr int BOX_BYTES = SSUB * spec::NBASIS * 8;             // bytes one TMA copy delivers
    static constexpr int ARR = (SSUB * spec::NBASIS + 15) / 16 * 16;      // slot stride per array (128-byte multiple)
    static constexpr int NTX = (spec::NA + TBX - 1) / TBX, NTY = (spec::NB + TBY - 1) / TBY;
    static constexpr int NITEMS = NTX * NTY * NZC;                        // work items: column x chunk
    static constexpr int PL = CZ + 2 * spec::RC;                          // planes staged per item
    static constexpr int NTHREADS = TBX * TBY * KZ;
    static_assert(RING >= LOOK + KZ + 2 * spec::RC && LOOK % KZ == 0, "ring too small for the look-ahead");
    static_assert((WX * 8) % 16 == 0, "TMA box rows must be multiples of 16 bytes");
};

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
__device__ __forceinline__ void tma_load_5d(u32 dst, const TensorMap *tm, int c0, int c1, int c2, int c3, int c4, u32 bar) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(bar) : "memory");
}

// partner of a cell in the staged ring: off[k][dz + RC] = index (in doubles, into smem) of the x component of the own CELL
// (sublattice 0) in the slot that holds lattice plane z + dz of array k
template <class G, int NCONF>
struct RingAcc {
    int off[NCONF][2 * spec::RC + 1];
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int k, double (&v)[3]) const {
        constexpr int O = BJ * Geo<G>::SSUB + DB * Geo<G>::SROW + DA;
        const double *q = smem + off[k][DC + spec::RC];
        v[0] = q[O]; v[1] = q[O + Geo<G>::WX]; v[2] = q[O + 2 * Geo<G>::WX];
    }
};

struct Item { int x0, y0, z0; };
template <class G>
__device__ __forceinline__ Item item_of(int j) {
    constexpr int NTX = Geo<G>::NTX, NTY = Geo<G>::NTY;
    const int item = (int)blockIdx.x + j * (int)gridDim.x;
    Item it;
    it.x0 = (item % NTX) * G::TBX;
    it.y0 = ((item / NTX) % NTY) * G::TBY;
    it.z0 = (item / (NTX * NTY)) * G::CZ;
    return it;
}

// one elected thread: start the copies of stream position q (plane p of this CTA's j-th item) for NARR arrays
template <class G, int NARR>
__device__ __forceinline__ void issue(int q, const TensorMap *const (&tm)[NARR], u32 bars) {
    constexpr int PL = Geo<G>::PL, ARR = Geo<G>::ARR, BOX_BYTES = Geo<G>::BOX_BYTES;
    const int j = q / PL, p = q - j * PL;
    const Item it = item_of<G>(j);
    const int slot = q % G::RING;
    const u32 bar = bars + 8u * slot;
    mbar_expect_tx(bar, (u32)(NARR * BOX_BYTES));
#pragma unroll
    for (int a = 0; a < NARR; ++a)
        tma_load_5d(smem_u32(smem + (slot * NARR + a) * ARR), tm[a], spec::LA + it.x0 - Geo<G>::HX, 0, spec::LB + it.y0 - spec::RB,
                    spec::LC + it.z0 - spec::RC + p, 0, bar);
}

// The marching loop shared by both sweeps: body(c, acc) is called once per thread and computed plane with
// acc.off[a][dz + RC] set for every staged array a.  KZ consecutive stream positions are computed per iteration, one per
// group of TBX*TBY threads (more warps per staged byte); LOOK is a multiple of KZ, RING >= LOOK + KZ + 2 RC.
template <class G, int NARR, class Body>
__device__ __forceinline__ void march(const TensorMap *const (&tm)[NARR], Body &&body) {
    constexpr int PL = Geo<G>::PL, ARR = Geo<G>::ARR, NITEMS = Geo<G>::NITEMS, SROW = Geo<G>::SROW, KZ = G::KZ, NT2 = G::TBX * G::TBY;
    u64 *bar_mem = (u64 *)(smem + G::RING * NARR * ARR);
    const u32 bars = smem_u32(bar_mem);
    const int tid = threadIdx.x;
    const int nmine = (NITEMS - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int Q = nmine * PL;
    if (tid == 0) {
        for (int s = 0; s < G::RING; ++s) mbar_init(bars + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0)
        for (int q = 0; q < G::LOOK && q < Q; ++q) issue<G, NARR>(q, tm, bars);
    const int kz = tid / NT2, t2 = tid - kz * NT2;
    const int txi = t2 % G::TBX, tyi = t2 / G::TBX;
    const int cell = (tyi + spec::RB) * SROW + (txi + Geo<G>::HX);
    for (int q0 = 0; q0 < Q; q0 += KZ) {
        if (tid == 0) {                                 // the slots of these positions were released by the barrier below
#pragma unroll
            for (int k = 0; k < KZ; ++k)
                if (q0 + G::LOOK + k < Q) issue<G, NARR>(q0 + G::LOOK + k, tm, bars);
        }
        const int q = q0 + kz;
        if (q < Q) {
            for (int k = 0; k <= kz; ++k) mbar_wait(bars + 8u * ((q0 + k) % G::RING), (u32)(((q0 + k) / G::RING) & 1));
            const int j = q / PL, p = q - j * PL;
            if (p >= 2 * spec::RC) {                   // planes z-RC .. z+RC of this item are staged: compute plane z
                const Item it = item_of<G>(j);
                Coord c;
                c.ia = it.x0 + txi; c.ib = it.y0 + tyi; c.ic = it.z0 + p - 2 * spec::RC;
                if (c.ia < spec::NA && c.ib < spec::NB && c.ic < spec::NC) {
                    RingAcc<G, NARR> acc;
#pragma unroll
                    for (int dz = -spec::RC; dz <= spec::RC; ++dz) {
                        const int slot = (q - spec::RC + dz) % G::RING;
#pragma unroll
                        for (int a = 0; a < NARR; ++a) acc.off[a][dz + spec::RC] = (slot * NARR + a) * ARR + cell;
                    }
                    body(c, acc);
                }
            }
        }
        __syncthreads();                               // every thread is done with the oldest planes: their slots may be refilled
    }
}

__device__ __forceinline__ int global_index(int b, const Coord &c) {
    return b * spec::SUB + (c.ic + spec::LC) * PLANE + (c.ib + spec::LB) * ROW + (c.ia + spec::LA);
}

}  // namespace spintma

extern "C" __global__ void __launch_bounds__(spintma::Geo<spec::TmaP>::NTHREADS)
    jit_predictor_tma(const __grid_constant__ spintma::TensorMap tm_n, const double *__restrict__ fddi, double *__restrict__ np,
                      const unsigned long long *__restrict__ d_step, unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi) {
    using namespace spintma;
    const u64 step = *d_step + step_add;
    const TensorMap *const tm[1] = {&tm_n};
    march<spec::TmaP, 1>(tm, [&](const Coord &c, const RingAcc<spec::TmaP, 1> &acc) {
        static_for<0, spec::NBASIS>([&](auto bb) {
            constexpr int B = decltype(bb)::value;
            const int idx = global_index(B, c);
            double own[1][3], F[1][3], sg[1][3] = {{0.0, 0.0, 0.0}};
            acc.template load<B, B, 0, 0, 0>(0, own[0]);
            thermal_force<B>(c, step, seed_lo, seed_hi, F[0]);
            force<B, 1>(acc, own, F);
            if constexpr (spec::HAS_DDI) { double d[3]; load3<0>(fddi + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
            if constexpr (spec::STT_ON) stt_gradient<B, 1>(acc, c, own, sg);
            double A[3], out[3];
            rotation_field<B>(own[0], F[0], sg[0], A);
            spin::rodrigues(A, specc::DT, specc::DT2, own[0], out);
            store_spin(np + idx, c, out);
        });
    });
}

extern "C" __global__ void __launch_bounds__(spintma::Geo<spec::TmaC>::NTHREADS)
    jit_corrector_tma(const __grid_constant__ spintma::TensorMap tm_n, const __grid_constant__ spintma::TensorMap tm_np,
                      const double *__restrict__ fddi_n, const double *__restrict__ fddi_np, double *__restrict__ nout,
                      const unsigned long long *__restrict__ d_step, unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi) {
    using namespace spintma;
    const u64 step = *d_step + step_add;
    const TensorMap *const tm[2] = {&tm_n, &tm_np};
    march<spec::TmaC, 2>(tm, [&](const Coord &c, const RingAcc<spec::TmaC, 2> &acc) {
        static_for<0, spec::NBASIS>([&](auto bb) {
            constexpr int B = decltype(bb)::value;
            const int idx = global_index(B, c);
            double th[3], A[3], Ap[3];
            thermal_force<B>(c, step, seed_lo, seed_hi, th);
            double own[2][3], F[2][3] = {{th[0], th[1], th[2]}, {th[0], th[1], th[2]}}, sg[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
            acc.template load<B, B, 0, 0, 0>(0, own[0]);
            acc.template load<B, B, 0, 0, 0>(1, own[1]);
            force<B, 2>(acc, own, F);
            if constexpr (spec::HAS_DDI) {
                double d[3];
                load3<0>(fddi_n + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2];
                load3<0>(fddi_np + idx, d); F[1][0] += d[0]; F[1][1] += d[1]; F[1][2] += d[2];
            }
            if constexpr (spec::STT_ON) stt_gradient<B, 2>(acc, c, own, sg);
            rotation_field<B>(own[0], F[0], sg[0], A);
            rotation_field<B>(own[1], F[1], sg[1], Ap);
            const double Ac[3] = {A[0] + Ap[0], A[1] + Ap[1], A[2] + Ap[2]};      // the 1/2 is folded into dt (exact)
            double out[3];
            spin::rodrigues(Ac, specc::HDT, specc::QDT2, own[0], out);
            spin::renormalise(out);
            store_spin(nout + idx, c, out);
        });
    });
}
