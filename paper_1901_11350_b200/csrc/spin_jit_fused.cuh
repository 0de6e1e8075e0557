// spin_jit_fused.cuh -- one Depondt step in ONE pass over the lattice (included by spin_jit_kernels.cuh when SPIN_FUSED is defined).
//
// The two-sweep step moves 120 B per spin-update through HBM (n -> n^p, then n^p and n -> n') and evaluates F(n) twice.  Here a
// block owns a tile of FTX x FTY x FTZ cells:
//   phase 1  predictor for the tile AND its rim of `reach` cells (the partners the corrector will gather): n^p goes to shared
//            memory, never to HBM; the rotation field A(n) of the tile's own cells (and their thermal field) is kept in shared
//            memory too, so F(n) is evaluated once;
//   phase 2  corrector for the tile's own cells: F(n^p) gathered from shared memory, A^c = (A + A^p)/2, n' = R(A^c) n, renormalise,
//            written to the other n buffer with its periodic images.
// HBM traffic: 48 B per spin-update (+ rim reads, which hit L2).  The price is the predictor work on the rim,
// (FTX+2r)(FTY+2r)(FTZ+2r)/(FTX FTY FTZ) = 1.66 for 32x8x8 at r = 1.  Rim cells compute exactly what the neighbouring block computes
// for them (same inputs, same code), so the result is bit-identical to the two-sweep kernels.
// A rim cell beyond a periodic edge is the wrapped lattice site (its own partners come from the ghost layers of n); beyond an open
// edge it is a zero vector, like the ghost layers.
//
// spec must define: FTX, FTY, FTZ (tile), FNT (threads per block).
#pragma once

namespace spinfused {
using namespace spinjit;

constexpr int WX = spec::FTX + 2 * spec::RA, WY = spec::FTY + 2 * spec::RB, WZ = spec::FTZ + 2 * spec::RC;      // tile + rim
constexpr int S_ROW = 3 * WX, S_PLANE = S_ROW * WY, S_SUB = S_PLANE * WZ;       // n^p in shared memory: [b][wz][wy][comp][wx]
constexpr int NP_DOUBLES = S_SUB * spec::NBASIS;
constexpr int T_ROW = 3 * spec::FTX, T_PLANE = T_ROW * spec::FTY, T_SUB = T_PLANE * spec::FTZ;   // A, noise: [b][tz][ty][comp][tx]
constexpr int A_DOUBLES = T_SUB * spec::NBASIS;
constexpr int NTX = (spec::NA + spec::FTX - 1) / spec::FTX, NTY = (spec::NB + spec::FTY - 1) / spec::FTY, NTZ = (spec::NC + spec::FTZ - 1) / spec::FTZ;

extern __shared__ __align__(16) double fsm[];      // [n^p : NP_DOUBLES][A : A_DOUBLES][thermal field : A_DOUBLES if THERMAL_ON]

// partner of a tile cell in the staged n^p: `cell` = index of the x component of the own CELL (sublattice 0)
struct TileAcc {
    int cell;
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int, double (&v)[3]) const {
        constexpr int O = BJ * S_SUB + DC * S_PLANE + DB * S_ROW + DA;
        const double *q = fsm + cell;
        v[0] = q[O]; v[1] = q[O + WX]; v[2] = q[O + 2 * WX];
    }
};

// wrap a coordinate that left the lattice through a periodic edge; false if it left through an open edge (or a ragged tile end)
template <int N, bool PER>
__device__ __forceinline__ bool wrap(int &x) {
    if (x >= 0 && x < N) return true;
    if constexpr (!PER) return false;
    else { x = x < 0 ? x + N : x - N; return x >= 0 && x < N; }
}

}  // namespace spinfused

extern "C" __global__ void __launch_bounds__(spec::FNT)
    jit_depondt_fused(const double *__restrict__ n, double *__restrict__ nout, const unsigned long long *__restrict__ d_step,
                      unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi, const unsigned char *__restrict__ pin) {
    using namespace spinfused;
    const u64 step = *d_step + step_add;
    int tile = blockIdx.x;
    const int x0 = (tile % NTX) * spec::FTX;
    tile /= NTX;
    const int y0 = (tile % NTY) * spec::FTY, z0 = (tile / NTY) * spec::FTZ;
    double *const s_np = fsm, *const s_A = fsm + NP_DOUBLES, *const s_th = fsm + NP_DOUBLES + A_DOUBLES;

    // ---- phase 1: predictor on the tile and its rim
    for (int s = threadIdx.x; s < WX * WY * WZ; s += spec::FNT) {
        const int wx = s % WX, wy = (s / WX) % WY, wz = s / (WX * WY);
        Coord c;
        c.ia = x0 + wx - spec::RA; c.ib = y0 + wy - spec::RB; c.ic = z0 + wz - spec::RC;
        const bool own_cell = wx >= spec::RA && wx < spec::RA + spec::FTX && wy >= spec::RB && wy < spec::RB + spec::FTY &&
                              wz >= spec::RC && wz < spec::RC + spec::FTZ;
        const bool exists = wrap<spec::NA, spec::PER_A>(c.ia) & wrap<spec::NB, spec::PER_B>(c.ib) & wrap<spec::NC, spec::PER_C>(c.ic);
        const int scell = wz * S_PLANE + wy * S_ROW + wx;
        const int tcell = (wz - spec::RC) * T_PLANE + (wy - spec::RB) * T_ROW + (wx - spec::RA);
        static_for<0, spec::NBASIS>([&](auto bb) {
            constexpr int B = decltype(bb)::value;
            double out[3] = {0.0, 0.0, 0.0};
            if (exists) {
                const int idx = B * spec::SUB + (c.ic + spec::LC) * PLANE + (c.ib + spec::LB) * ROW + (c.ia + spec::LA);
                GlobalAcc<1> cfg;
                cfg.cfg[0] = n + idx;
                double own[1][3], F[1][3], sg[1][3] = {{0.0, 0.0, 0.0}};
                load3<0>(cfg.cfg[0], own[0]);
                if (is_pinned<B>(pin, c)) {
                    out[0] = own[0][0]; out[1] = own[0][1]; out[2] = own[0][2];
                } else {
                    thermal_force<B>(c, step, seed_lo, seed_hi, F[0]);
                    if constexpr (spec::THERMAL_ON) {
                        if (own_cell) { double *t = s_th + B * T_SUB + tcell; t[0] = F[0][0]; t[spec::FTX] = F[0][1]; t[2 * spec::FTX] = F[0][2]; }
                    }
                    force<B, 1>(cfg, own, F);
                    if constexpr (spec::STT_ON) stt_gradient<B, 1>(cfg, c, own, sg);
                    double A[3];
                    rotation_field<B>(own[0], F[0], sg[0], A);
                    spin::rodrigues(A, specc::DT, specc::DT2, own[0], out);
                    if (own_cell) { double *a = s_A + B * T_SUB + tcell; a[0] = A[0]; a[spec::FTX] = A[1]; a[2 * spec::FTX] = A[2]; }
                }
            }
            double *q = s_np + B * S_SUB + scell;
            q[0] = out[0]; q[WX] = out[1]; q[2 * WX] = out[2];
        });
    }
    __syncthreads();

    // ---- phase 2: corrector on the tile's own cells
    for (int s = threadIdx.x; s < spec::FTX * spec::FTY * spec::FTZ; s += spec::FNT) {
        const int tx = s % spec::FTX, ty = (s / spec::FTX) % spec::FTY, tz = s / (spec::FTX * spec::FTY);
        Coord c;
        c.ia = x0 + tx; c.ib = y0 + ty; c.ic = z0 + tz;
        if (c.ia >= spec::NA || c.ib >= spec::NB || c.ic >= spec::NC) continue;
        TileAcc acc;
        acc.cell = (tz + spec::RC) * S_PLANE + (ty + spec::RB) * S_ROW + (tx + spec::RA);
        const int tcell = tz * T_PLANE + ty * T_ROW + tx;
        static_for<0, spec::NBASIS>([&](auto bb) {
            constexpr int B = decltype(bb)::value;
            const int idx = B * spec::SUB + (c.ic + spec::LC) * PLANE + (c.ib + spec::LB) * ROW + (c.ia + spec::LA);
            double n0[3];
            load3<0>(n + idx, n0);
            if (is_pinned<B>(pin, c)) { store_spin(nout + idx, c, n0); return; }
            double own[1][3], F[1][3] = {{-0.0, -0.0, -0.0}}, sg[1][3] = {{0.0, 0.0, 0.0}}, A[3], Ap[3];
            if constexpr (spec::THERMAL_ON) { const double *t = s_th + B * T_SUB + tcell; F[0][0] = t[0]; F[0][1] = t[spec::FTX]; F[0][2] = t[2 * spec::FTX]; }
            acc.template load<B, B, 0, 0, 0>(0, own[0]);
            force<B, 1>(acc, own, F);
            if constexpr (spec::STT_ON) stt_gradient<B, 1>(acc, c, own, sg);
            rotation_field<B>(own[0], F[0], sg[0], Ap);
            { const double *a = s_A + B * T_SUB + tcell; A[0] = a[0]; A[1] = a[spec::FTX]; A[2] = a[2 * spec::FTX]; }
            const double Ac[3] = {A[0] + Ap[0], A[1] + Ap[1], A[2] + Ap[2]};      // the 1/2 is folded into dt (exact)
            double out[3];
            spin::rodrigues(Ac, specc::HDT, specc::QDT2, n0, out);
            spin::renormalise(out);
            store_spin(nout + idx, c, out);
        });
    }
}
