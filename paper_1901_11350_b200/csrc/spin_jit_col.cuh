// spin_jit_col.cuh -- the two Depondt sweeps as column-marching kernels (included by spin_jit_kernels.cuh when SPIN_COL is defined).
//
// Why (profiles/r1c_README.md): the brick kernels are bound by the L1 data pipe -- 67 LSU wavefronts per warp for the 21 vector
// loads + 3 stores of a nearest-neighbour stencil, 5.6 bytes through L1 per byte of HBM traffic -- and shared-memory staging
// (spin_jit_tma.cuh) moves the same wavefronts to the same pipe.  The only way to take wavefronts away is to reuse a loaded
// spin from registers: here one thread owns a lattice column (ia, ib) and marches along c through a chunk of CCZ planes,
// keeping its own spin at z-1, z, z+1 in registers.  The partners at (0, 0, +-1) of the own sublattice then cost nothing, and
// the own spin is loaded once instead of three times: 15 vector loads per site instead of 21 (30 instead of 42 in the corrector).
// Everything else (gather table, arithmetic, ghost images, noise) is the code of the brick kernels.
//
// Needs a ghost plane below and above (spec::RC >= 1) and spec::NC >= 2; spec must define CBX, CBY (column tile), CCZ (planes
// per chunk), CNZC (chunks).
#pragma once

namespace spincol {
using namespace spinjit;

template <int NCONF>
struct ColAcc {
    const double *cfg[NCONF];      // x component of the own site (current plane) in configuration k
    double zr[NCONF][3][3];        // own column in registers: [k][dz + 1][component]
    template <int B, int BJ, int DA, int DB, int DC>
    __device__ __forceinline__ void load(int k, double (&v)[3]) const {
        if constexpr (BJ == B && DA == 0 && DB == 0 && DC >= -1 && DC <= 1) {
            v[0] = zr[k][DC + 1][0]; v[1] = zr[k][DC + 1][1]; v[2] = zr[k][DC + 1][2];
        } else {
            load3<lin<B, BJ, DA, DB, DC>()>(cfg[k], v);
        }
    }
    __device__ __forceinline__ void advance() {      // z -> z + 1: shift the register window, move the pointers one plane up
#pragma unroll
        for (int k = 0; k < NCONF; ++k) {
#pragma unroll
            for (int c = 0; c < 3; ++c) { zr[k][0][c] = zr[k][1][c]; zr[k][1][c] = zr[k][2][c]; }
            cfg[k] += PLANE;
        }
    }
};

constexpr int NTX = (spec::NA + spec::CBX - 1) / spec::CBX, NTY = (spec::NB + spec::CBY - 1) / spec::CBY;

// column of this thread: lattice coordinates of its first site, index of that site, number of planes; false if outside
template <int B>
__device__ __forceinline__ bool locate_column(Coord &c, int &idx, int &nz) {
    int item = blockIdx.x;
    const int tx = item % NTX;
    item /= NTX;
    const int ty = item % NTY, zc = item / NTY;
    const int t = threadIdx.x;
    c.ia = tx * spec::CBX + (t % spec::CBX);
    c.ib = ty * spec::CBY + (t / spec::CBX);
    c.ic = zc * spec::CCZ;
    nz = spec::NC - c.ic < spec::CCZ ? spec::NC - c.ic : spec::CCZ;
    idx = B * spec::SUB + (c.ic + spec::LC) * PLANE + (c.ib + spec::LB) * ROW + (c.ia + spec::LA);
    return (c.ia < spec::NA) && (c.ib < spec::NB) && nz > 0;
}

template <int B>
__device__ __forceinline__ void predictor_column(const double *__restrict__ n, const double *__restrict__ fddi, double *__restrict__ np,
                                                 u64 step, u32 seed_lo, u32 seed_hi) {
    Coord c;
    int idx, nz;
    if (!locate_column<B>(c, idx, nz)) return;
    ColAcc<1> acc;
    acc.cfg[0] = n + idx;
    load3<-PLANE>(acc.cfg[0], acc.zr[0][0]);
    load3<0>(acc.cfg[0], acc.zr[0][1]);
    for (int z = 0; z < nz; ++z) {
        load3<PLANE>(acc.cfg[0], acc.zr[0][2]);
        double own[1][3] = {{acc.zr[0][1][0], acc.zr[0][1][1], acc.zr[0][1][2]}}, F[1][3], sg[1][3] = {{0.0, 0.0, 0.0}};
        thermal_force<B>(c, step, seed_lo, seed_hi, F[0]);
        force<B, 1>(acc, own, F);
        if constexpr (spec::HAS_DDI) { double d[3]; load3<0>(fddi + idx, d); F[0][0] += d[0]; F[0][1] += d[1]; F[0][2] += d[2]; }
        if constexpr (spec::STT_ON) stt_gradient<B, 1>(acc, c, own, sg);
        double A[3], out[3];
        rotation_field<B>(own[0], F[0], sg[0], A);
        spin::rodrigues(A, specc::DT, specc::DT2, own[0], out);
        store_spin(np + idx, c, out);
        acc.advance();
        idx += PLANE;
        c.ic += 1;
    }
}

template <int B>
__device__ __forceinline__ void corrector_column(const double *__restrict__ n, const double *__restrict__ np, const double *__restrict__ fddi_n,
                                                 const double *__restrict__ fddi_np, double *__restrict__ nout, u64 step, u32 seed_lo, u32 seed_hi) {
    Coord c;
    int idx, nz;
    if (!locate_column<B>(c, idx, nz)) return;
    ColAcc<2> acc;
    acc.cfg[0] = n + idx;
    acc.cfg[1] = np + idx;
#pragma unroll
    for (int k = 0; k < 2; ++k) { load3<-PLANE>(acc.cfg[k], acc.zr[k][0]); load3<0>(acc.cfg[k], acc.zr[k][1]); }
    for (int z = 0; z < nz; ++z) {
        load3<PLANE>(acc.cfg[0], acc.zr[0][2]);
        load3<PLANE>(acc.cfg[1], acc.zr[1][2]);
        double th[3], A[3], Ap[3];
        thermal_force<B>(c, step, seed_lo, seed_hi, th);
        double own[2][3] = {{acc.zr[0][1][0], acc.zr[0][1][1], acc.zr[0][1][2]}, {acc.zr[1][1][0], acc.zr[1][1][1], acc.zr[1][1][2]}};
        double F[2][3] = {{th[0], th[1], th[2]}, {th[0], th[1], th[2]}}, sg[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
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
        acc.advance();
        idx += PLANE;
        c.ic += 1;
    }
}

}  // namespace spincol

extern "C" __global__ void SPIN_BOUNDS(spec::CBX *spec::CBY)
    jit_predictor_col(const double *__restrict__ n, const double *__restrict__ fddi, double *__restrict__ np,
                      const unsigned long long *__restrict__ d_step, unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi) {
    const unsigned long long step = *d_step + step_add;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        spincol::predictor_column<decltype(b)::value>(n, fddi, np, step, seed_lo, seed_hi);
    });
}

extern "C" __global__ void SPIN_BOUNDS(spec::CBX *spec::CBY)
    jit_corrector_col(const double *__restrict__ n, const double *__restrict__ np, const double *__restrict__ fddi_n,
                      const double *__restrict__ fddi_np, double *__restrict__ nout, const unsigned long long *__restrict__ d_step,
                      unsigned int step_add, unsigned int seed_lo, unsigned int seed_hi) {
    const unsigned long long step = *d_step + step_add;
    spinjit::dispatch_basis<0>((int)blockIdx.y, [&](auto b) {
        spincol::corrector_column<decltype(b)::value>(n, np, fddi_n, fddi_np, nout, step, seed_lo, seed_hi);
    });
}
