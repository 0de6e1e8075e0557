// spin_jit.cu -- run-time specialisation of the two Depondt sweeps (spin_jit_kernels.cuh) with NVRTC.
//
// The device plan of a system (gather tables, lattice extents, LLG prefactors) is printed as `constexpr` data into
// `namespace spec`, followed by `#include "spin_jit_kernels.cuh"`; NVRTC compiles that translation unit for sm_100a and the
// cubin is loaded through the runtime's library API.  The result is cached per system and rebuilt when the plan changes.
// If NVRTC is unavailable or compilation fails the system keeps using the table-driven kernels and records why
// (spin_kernel_info reports which path is active; nothing is silently computed on the CPU either way).
#include <cuda.h>
#include <dlfcn.h>
#include <nvrtc.h>
#include <stdlib.h>
#include <stdio.h>
#include <stddef.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <vector>
#include <mutex>
#include <sstream>
#include <string>

#include "spinllg_internal.h"

using namespace spin;

// staging geometry of one TMA-fed sweep (spin_jit_tma.cuh): tile, ring depth, look-ahead, chunks along c
struct TmaGeo {
    int tbx, tby, kz, ring, look, nzc, cz;
    int narr;                 // arrays staged per plane (predictor 1, corrector 2)
    size_t smem_bytes;
    int items;
};

struct JitState {
    cudaLibrary_t lib;
    cudaKernel_t k_pred, k_corr, k_rk4;
    bool loaded;
    std::string source, log;
    // TMA-fed plane-marching sweeps
    bool tma;                 // generated and loaded
    std::string tma_note;     // why not, if not
    TmaGeo gp, gc;
    cudaKernel_t k_pred_tma, k_corr_tma;
    // one-pass Depondt step (spin_jit_fused.cuh)
    bool fused;
    cudaKernel_t k_fused;
    int fused_geo[4];         // FTX, FTY, FTZ, FNT
    size_t fused_smem;
    // all steps in one cooperative launch (launch-bound lattices)
    bool coop;
    cudaKernel_t k_coop;
    int coop_grid;
    bool cluster;             // the whole lattice is one thread-block cluster (<= 16 bricks): hardware barrier instead of the grid barrier
    cudaKernel_t k_cluster;
    // column-marching sweeps
    bool col;
    cudaKernel_t k_pred_col, k_corr_col;
    int col_geo[4];           // CBX, CBY, CCZ, CNZC
    // two sites per thread, 128-bit accesses (spin_jit_pair.cuh)
    bool pair;
    cudaKernel_t k_pred_pair, k_corr_pair;
    int pair_geo[3];          // VBX, VBY, VBZ
    int grid_p, grid_c;
    CUtensorMap tm_n[2];              // predictor: n[cur] with the predictor tile
    CUtensorMap tm_cn[2], tm_cnp;     // corrector: n[cur], n^p with the corrector tile
};

namespace {

std::string hexd(double v) {
    char buf[64];
    if (v == 0.0) return "0.0";
    snprintf(buf, sizeof(buf), "%a", v);       // exact hexadecimal floating literal (C++17)
    return buf;
}

std::string csrc_dir() {
    Dl_info info;
    if (dladdr((void *)&spin::jit_release, &info) && info.dli_fname) {
        std::string p(info.dli_fname);
        const size_t k = p.find_last_of('/');
        return (k == std::string::npos ? std::string(".") : p.substr(0, k)) + "/csrc";
    }
    return "csrc";
}

template <class T, class F>
void emit_array(std::ostringstream &o, const char *type, const char *name, int n, F &&get) {
    o << "constexpr " << type << " " << name << "[" << (n > 0 ? n : 1) << "] = {";
    for (int i = 0; i < n; ++i) o << (i ? ", " : "") << get(i);
    if (n == 0) o << "0";
    o << "};\n";
}

}  // namespace

namespace {

int sm_count(const spin_system *s) {
    int n = 148;
    if (s->has_device) { int dev = 0; if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev); }
    return n > 0 ? n : 148;
}

// Choose the staging geometry of one sweep.  Defaults: 32 x TBY tiles (TBY 8), look-ahead 3 planes; the number of chunks along
// c is chosen so that the work items fill the resident CTAs evenly while the 2*rC extra planes per chunk stay cheap.
// SPINLLG_TMA_P / SPINLLG_TMA_C = "tbx,tby,look,nzc,kz" override (0 = default) for tuning.
bool plan_tma_geo(const spin_system *s, int narr, const char *env, TmaGeo &g, std::string &why) {
    const DevicePlan &P = s->plan;
    int tbx = 32, tby = 8, look = 2, nzc = 0, kz = 2;
    if (const char *e = getenv(env)) {
        int v[5] = {0, 0, 0, 0, 0};
        sscanf(e, "%d,%d,%d,%d,%d", &v[0], &v[1], &v[2], &v[3], &v[4]);
        if (v[0] > 0) tbx = v[0];
        if (v[1] > 0) tby = v[1];
        if (v[2] > 0) look = v[2];
        if (v[3] > 0) nzc = v[3];
        if (v[4] > 0) kz = v[4];
    }
    look = (look + kz - 1) / kz * kz;
    if (tbx % 2 || (tbx * tby) % 32 || tbx * tby * kz > 1024) { why = "tile must have an even width and a multiple of 32 cells, at most 1024 threads"; return false; }
    g.tbx = tbx; g.tby = tby; g.kz = kz; g.look = look; g.ring = look + kz + 2 * P.rC; g.narr = narr;
    const int wx = tbx + 2 * ((P.rA + 1) / 2 * 2), wy = tby + 2 * P.rB;      // rim along a rounded up to even (16-byte aligned box rows)
    if (wx > 256 || wy > 256 || P.nb > 256) { why = "staged box exceeds the TMA box limit of 256 per dimension"; return false; }
    const size_t arr = ((size_t)3 * wx * wy * P.nb + 15) / 16 * 16;
    g.smem_bytes = (size_t)g.ring * narr * arr * 8 + (size_t)g.ring * 8;
    if (g.smem_bytes > 220 * 1024) { why = "staging ring does not fit in shared memory"; return false; }
    const int cols = ((P.Na + tbx - 1) / tbx) * ((P.Nb + tby - 1) / tby);
    int per_sm = (int)std::min<size_t>((size_t)2048 / (tbx * tby * kz), (size_t)(227 * 1024) / (g.smem_bytes + 1024));
    if (per_sm < 1) per_sm = 1;
    const int slots = sm_count(s) * per_sm;
    if (nzc <= 0) {
        double best = -1.0;
        for (int k = 1; k <= P.Nc; ++k) {
            const int cz = (P.Nc + k - 1) / k;
            if ((k - 1) * cz >= P.Nc) continue;                           // an empty last chunk
            const long items = (long)cols * k;
            const long waves = (items + slots - 1) / slots;
            const double util = (double)items / (double)(waves * slots);
            const double eff = util * (double)P.Nc / ((double)k * (cz + 2 * P.rC));
            if (eff > best + 1e-9) { best = eff; nzc = k; }
        }
    }
    if (nzc > P.Nc) nzc = P.Nc;
    g.nzc = nzc; g.cz = (P.Nc + nzc - 1) / nzc;
    g.items = cols * nzc;
    return true;
}

void emit_tma_geo(std::ostringstream &o, const char *name, const TmaGeo &g) {
    o << "struct " << name << " { static constexpr int TBX = " << g.tbx << ", TBY = " << g.tby << ", KZ = " << g.kz << ", RING = " << g.ring << ", LOOK = " << g.look
      << ", NZC = " << g.nzc << ", CZ = " << g.cz << "; };\n";
}

}  // namespace

// brick of the specialised brick kernels: BX x BY x BZ sites per block (SPINLLG_BRICK="bx,by,bz" overrides, for tuning)
static void jit_brick(const spin_system *s, int b[3]) {
    const bool flat = s->nc[2] < 2;
    b[0] = 32; b[1] = flat ? 8 : 4; b[2] = flat ? 1 : 2;
    if (const char *e = getenv("SPINLLG_BRICK")) {
        int v[3] = {0, 0, 0};
        sscanf(e, "%d,%d,%d", &v[0], &v[1], &v[2]);
        if (v[0] > 0 && v[1] > 0 && v[2] > 0 && v[0] * v[1] * v[2] <= 1024 && (v[0] * v[1] * v[2]) % 32 == 0 && (!flat || v[2] == 1)) { b[0] = v[0]; b[1] = v[1]; b[2] = v[2]; }
    }
}
static void jit_brick_launch(const spin_system *s, dim3 &grid, dim3 &block);
// programmatic dependent launch of the brick sweeps: 0 off, 1 dependents released at entry, 2 at the end of each block.
// Measured (profiles/r1g_README.md): sweeps of many waves gain 1-3 % from 1 and lose with 2.  Sweeps of about one wave lose with 1 (the
// next sweep's blocks are placed while this one's still hold their SMs, unevenly); with 2 they gain 10-14 % when the kernels were
// compiled by NVRTC 12.9 and lose 4 % with NVRTC 12.8, so the automatic choice depends on the compiler that was found.
static bool nvrtc_at_least(int major, int minor);
static int pdl_mode(const spin_system *s) {
    if (s->opt_pdl >= 0) return s->opt_pdl;
    dim3 grid, block;
    jit_brick_launch(s, grid, block);
    const long blocks = (long)grid.x * grid.y * s->n_img;
    if (blocks > 6L * sm_count(s)) return 1;
    return nvrtc_at_least(12, 9) ? 2 : 0;
}
static void jit_brick_launch(const spin_system *s, dim3 &grid, dim3 &block) {
    int b[3];
    jit_brick(s, b);
    grid = dim3((unsigned)(((s->nc[0] + b[0] - 1) / b[0]) * ((s->nc[1] + b[1] - 1) / b[1]) * ((s->nc[2] + b[2] - 1) / b[2])), (unsigned)s->nb, 1);
    block = dim3((unsigned)(b[0] * b[1] * b[2]), 1, 1);
}

// one-pass Depondt step (spin_jit_fused.cuh): tile and threads per block, shared-memory bytes; false if not applicable.
// SPINLLG_FUSED="ftx,fty,ftz,threads" overrides the defaults (32 x 8 x 8 cells, 512 threads; flat lattices 32 x 16 x 1).
static bool plan_fused(const spin_system *s, int g[4], size_t &smem) {
    const DevicePlan &P = s->plan;
    if (!s->opt_fused || s->solver != 0 || s->ddi_on || s->opt_store_A || s->n_img > 1) return false;
    if (s->opt_fused < 2 && s->N < 16384) return false;
    const bool flat = P.Nc < 2;
    int v[4] = {32, flat ? 16 : 8, flat ? 1 : 8, 512};
    if (const char *e = getenv("SPINLLG_FUSED")) {
        int u[4] = {0, 0, 0, 0};
        sscanf(e, "%d,%d,%d,%d", &u[0], &u[1], &u[2], &u[3]);
        for (int k = 0; k < 4; ++k) if (u[k] > 0) v[k] = u[k];
    }
    if (v[2] > P.Nc) v[2] = P.Nc;
    if (v[3] % 32 || v[3] > 1024) return false;
    const size_t np = (size_t)3 * (v[0] + 2 * P.rA) * (v[1] + 2 * P.rB) * (v[2] + 2 * P.rC) * P.nb;
    const size_t a = (size_t)3 * v[0] * v[1] * v[2] * P.nb;
    smem = (np + a * (P.thermal_on ? 2 : 1)) * sizeof(double);
    if (smem > 220 * 1024) return false;
    for (int k = 0; k < 4; ++k) g[k] = v[k];
    return true;
}

// column-marching sweeps (spin_jit_col.cuh): tile of columns per block, planes per chunk, chunks; false if not applicable.
// SPINLLG_COL="cbx,cby,ccz" overrides the defaults (32 x 4 columns, 16 planes per chunk).
static bool plan_col(const spin_system *s, int g[4]) {
    const DevicePlan &P = s->plan;
    if (!s->opt_col || s->opt_store_A || s->solver != 0 || s->d_pin || s->n_img > 1 || P.rC < 1 || P.Nc < 2) return false;
    int cbx = 32, cby = 4, ccz = 16;
    if (const char *e = getenv("SPINLLG_COL")) {
        int v[3] = {0, 0, 0};
        sscanf(e, "%d,%d,%d", &v[0], &v[1], &v[2]);
        if (v[0] > 0) cbx = v[0];
        if (v[1] > 0) cby = v[1];
        if (v[2] > 0) ccz = v[2];
    }
    if ((cbx * cby) % 32 || cbx * cby > 1024) return false;
    if (ccz > P.Nc) ccz = P.Nc;
    g[0] = cbx; g[1] = cby; g[2] = ccz; g[3] = (P.Nc + ccz - 1) / ccz;
    return true;
}

// two sites per thread (spin_jit_pair.cuh): brick of sites per block; false if not applicable (odd rows, options the variant does not
// carry).  SPINLLG_PAIR="vbx,vby,vbz" overrides the default brick (32 x 4 x 2 sites = 128 threads).
static bool plan_pair(const spin_system *s, int g[3]) {
    const DevicePlan &P = s->plan;
    if (!s->opt_pair || s->opt_store_A || s->solver != 0 || s->d_pin || s->n_img > 1) return false;
    if (P.Na % 2 || P.LA % 2 || P.PA % 2 || P.sub % 2) return false;
    int v[3] = {32, 4, 2};
    if (const char *e = getenv("SPINLLG_PAIR")) {
        int w[3] = {0, 0, 0};
        sscanf(e, "%d,%d,%d", &w[0], &w[1], &w[2]);
        for (int k = 0; k < 3; ++k) if (w[k] > 0) v[k] = w[k];
    }
    if (P.Nc == 1) { v[1] *= v[2]; v[2] = 1; }
    while (v[0] > 2 && v[0] / 2 >= P.Na) { v[0] /= 2; v[1] *= 2; }      // short rows: same threads, more rows per block
    const int threads = v[0] / 2 * v[1] * v[2];
    if (v[0] % 2 || threads % 32 || threads > 1024) return false;
    g[0] = v[0]; g[1] = v[1]; g[2] = v[2];
    return true;
}

// the staging geometry of both sweeps, or why the TMA-fed sweeps are not generated for this system
static bool plan_tma(const spin_system *s, TmaGeo &gp, TmaGeo &gc, std::string &why) {
    if (!s->opt_tma) { why = "disabled by option use_tma=0"; return false; }
    if (s->solver != 0) { why = "Depondt solver only"; return false; }
    if (s->d_pin) { why = "pinned spins use the brick kernels"; return false; }
    if (s->n_img > 1) { why = "batched images use the brick kernels"; return false; }
    if (s->opt_store_A) { why = "store_A=1 uses the brick kernels"; return false; }
    if (s->opt_tma < 2 && s->N < 16384) { why = "lattice too small to fill persistent CTAs"; return false; }
    return plan_tma_geo(s, 1, "SPINLLG_TMA_P", gp, why) && plan_tma_geo(s, 2, "SPINLLG_TMA_C", gc, why);
}

std::string spin::jit_source(const spin_system *s) {
    const DevicePlan &P = s->plan;
    std::ostringstream o;
    
    o << "// generated by spin_jit.cu -- one spin system as compile-time constants\n";
    o << "namespace spec {\n";
    o << "constexpr int NA = " << P.Na << ", NB = " << P.Nb << ", NC = " << P.Nc << ", NBASIS = " << P.nb << ";\n";
    o << "constexpr int LA = " << P.LA << ", LB = " << P.LB << ", LC = " << P.LC << ", PA = " << P.PA << ", PB = " << P.PB << ", PC = " << P.PC
      << ", SUB = " << P.sub << ", RA = " << P.rA << ", RB = " << P.rB << ", RC = " << P.rC << ";\n";
    o << "constexpr bool GA = " << (P.gA ? "true" : "false") << ", GB = " << (P.gB ? "true" : "false") << ", GC = "
      << (P.gC ? "true" : "false") << ";\n";
    int brick[3];
    jit_brick(s, brick);
    o << "constexpr int BX = " << brick[0] << ", BY = " << brick[1] << ", BZ = " << brick[2] << ";\n";
    o << "constexpr bool PER_A = " << (P.perA ? "true" : "false") << ", PER_B = " << (P.perB ? "true" : "false")
      << ", PER_C = " << (P.perC ? "true" : "false") << ";\n";
    o << "constexpr bool CACHE_NOISE = " << ((s->opt_cache_noise && P.thermal_on && !(s->opt_store_A && s->solver == 0)) ? "true" : "false") << ";\n";
    {   // corrector: the fields of n and of n^p one after the other (40 registers, 1.5 % faster on cfg3) or interleaved (48)
        const char *e = getenv("SPINLLG_SPLIT");
        o << "constexpr bool SPLIT_CORR = " << ((e && atoi(e) == 0) ? "false" : "true") << ";\n";
    }
    {   // corrector bricks in reverse order (L2 reuse of what the predictor touched last): 68.1 -> 65.3 us per step on cfg3
        const char *e = getenv("SPINLLG_REVERSE");
        o << "constexpr bool REVERSE_CORR = " << ((e && atoi(e) == 0) ? "false" : "true") << ";\n";
    }
    // programmatic dependent launch: the sweeps release their dependents at once and wait for their prerequisites in the kernel
    o << "constexpr int PDL = " << pdl_mode(s) << ";      // 0 off, 1 dependents released at entry, 2 at the end of the block\n";
    o << "constexpr bool MULTI_IMAGE = " << (s->n_img > 1 ? "true" : "false") << ";\n";
    o << "constexpr bool DAMPING_ONLY = " << (s->damping_only ? "true" : "false") << ";\n";
    o << "constexpr bool HAS_PIN = " << (s->d_pin ? "true" : "false") << ";\n";
    o << "constexpr int SOLVER = " << s->solver << ";      // 0 Depondt, 1 Heun, 2 SIB, 3 RK4 (own stage kernel)\n";
    o << "constexpr bool STORE_A = " << ((s->opt_store_A && s->solver == 0) ? "true" : "false") << ", HAS_DDI = " << (P.has_ddi ? "true" : "false")
      << ", THERMAL_ON = " << (P.thermal_on ? "true" : "false") << ", STT_ON = " << (P.stt_on ? "true" : "false") << ";\n";
    const int np = P.pair_begin[P.nb], nq = P.quad_begin[P.nb];
    emit_array<int>(o, "int", "PAIR_BEGIN", P.nb + 1, [&](int i) { return std::to_string(P.pair_begin[i]); });
    emit_array<int>(o, "int", "P_DA", np, [&](int i) { return std::to_string(P.pairs[i].da); });
    emit_array<int>(o, "int", "P_DB", np, [&](int i) { return std::to_string(P.pairs[i].db); });
    emit_array<int>(o, "int", "P_DC", np, [&](int i) { return std::to_string(P.pairs[i].dc); });
    emit_array<int>(o, "int", "P_BJ", np, [&](int i) { return std::to_string(P.pairs[i].bj); });
    emit_array<double>(o, "double", "P_J", np, [&](int i) { return hexd(P.pairs[i].J); });
    emit_array<double>(o, "double", "P_DX", np, [&](int i) { return hexd(P.pairs[i].Dx); });
    emit_array<double>(o, "double", "P_DY", np, [&](int i) { return hexd(P.pairs[i].Dy); });
    emit_array<double>(o, "double", "P_DZ", np, [&](int i) { return hexd(P.pairs[i].Dz); });
    emit_array<int>(o, "int", "QUAD_BEGIN", P.nb + 1, [&](int i) { return std::to_string(P.quad_begin[i]); });
    o << "constexpr int Q_D[" << (nq ? nq : 1) << "][9] = {";
    for (int i = 0; i < nq; ++i) {
        o << (i ? ", {" : "{");
        for (int m = 0; m < 3; ++m) for (int d = 0; d < 3; ++d) o << ((m || d) ? ", " : "") << P.quads[i].d[m][d];
        o << "}";
    }
    if (!nq) o << "{0, 0, 0, 0, 0, 0, 0, 0, 0}";
    o << "};\n";
    o << "constexpr int Q_B[" << (nq ? nq : 1) << "][3] = {";
    for (int i = 0; i < nq; ++i) o << (i ? ", {" : "{") << P.quads[i].b[0] << ", " << P.quads[i].b[1] << ", " << P.quads[i].b[2] << "}";
    if (!nq) o << "{0, 0, 0}";
    o << "};\n";
    emit_array<double>(o, "double", "Q_K", nq, [&](int i) { return hexd(P.quads[i].K); });
    auto emit_b3 = [&](const char *name, const double (*v)[3]) {
        o << "constexpr double " << name << "[" << P.nb << "][3] = {";
        for (int b = 0; b < P.nb; ++b) o << (b ? ", {" : "{") << hexd(v[b][0]) << ", " << hexd(v[b][1]) << ", " << hexd(v[b][2]) << "}";
        o << "};\n";
    };
    emit_b3("ZEE", P.zee);
    const int na = P.ani_begin[P.nb];
    emit_array<int>(o, "int", "ANI_BEGIN", P.nb + 1, [&](int i) { return std::to_string(P.ani_begin[i]); });
    o << "constexpr double KAX[" << (na ? na : 1) << "][3] = {";
    for (int e = 0; e < na; ++e) o << (e ? ", {" : "{") << hexd(P.Kax[e][0]) << ", " << hexd(P.Kax[e][1]) << ", " << hexd(P.Kax[e][2]) << "}";
    if (!na) o << "{0.0, 0.0, 0.0}";
    o << "};\n";
    emit_array<double>(o, "double", "K2", na, [&](int i) { return hexd(P.K2[i]); });
    emit_array<double>(o, "double", "PRE", P.nb, [&](int i) { return hexd(P.pre[i]); });
    emit_array<double>(o, "double", "SIGMA", P.nb, [&](int i) { return hexd(P.sigma[i]); });
    o << "constexpr double ALPHA = " << hexd(P.alpha) << ", DT = " << hexd(P.dt) << ", DT2 = " << hexd(P.dt2) << ";\n";
    o << "constexpr double STT_C[3] = {" << hexd(P.stt_on ? P.stt_c[0] : 0.0) << ", " << hexd(P.stt_on ? P.stt_c[1] : 0.0) << ", "
      << hexd(P.stt_on ? P.stt_c[2] : 0.0) << "};\n";
    o << "constexpr double STT_S = " << hexd(P.stt_s) << ", STT_X = " << hexd(P.stt_x) << ";\n";
    // the same values in constant memory (operands of the fp64 instructions; spec:: decides at compile time what is zero)
    o << "}  // namespace spec\nnamespace specc {\n";
    auto emit_c = [&](const char *name, int n, auto &&get) {
        o << "__constant__ double " << name << "[" << (n > 0 ? n : 1) << "] = {";
        for (int i = 0; i < n; ++i) o << (i ? ", " : "") << hexd(get(i));
        if (n == 0) o << "0.0";
        o << "};\n";
    };
    auto emit_cb3 = [&](const char *name, const double (*v)[3]) {
        o << "__constant__ double " << name << "[" << P.nb << "][3] = {";
        for (int b = 0; b < P.nb; ++b) o << (b ? ", {" : "{") << hexd(v[b][0]) << ", " << hexd(v[b][1]) << ", " << hexd(v[b][2]) << "}";
        o << "};\n";
    };
    emit_c("P_J", np, [&](int i) { return P.pairs[i].J; });
    emit_c("P_DX", np, [&](int i) { return P.pairs[i].Dx; });
    emit_c("P_DY", np, [&](int i) { return P.pairs[i].Dy; });
    emit_c("P_DZ", np, [&](int i) { return P.pairs[i].Dz; });
    emit_c("Q_K", nq, [&](int i) { return P.quads[i].K; });
    emit_cb3("ZEE", P.zee);
    o << "__constant__ double KAX[" << (na ? na : 1) << "][3] = {";
    for (int e = 0; e < na; ++e) o << (e ? ", {" : "{") << hexd(P.Kax[e][0]) << ", " << hexd(P.Kax[e][1]) << ", " << hexd(P.Kax[e][2]) << "}";
    if (!na) o << "{0.0, 0.0, 0.0}";
    o << "};\n";
    emit_c("K2", na, [&](int i) { return P.K2[i]; });
    emit_c("PRE", P.nb, [&](int i) { return P.pre[i]; });
    emit_c("PREA", P.nb, [&](int i) { return P.pre[i] * P.alpha; });
    emit_c("SIGMA", P.nb, [&](int i) { return P.sigma[i]; });
    emit_c("STT_C", 3, [&](int i) { return P.stt_on ? P.stt_c[i] : 0.0; });
    o << "__constant__ double DT = " << hexd(P.dt) << ", DT2 = " << hexd(P.dt2) << ", HDT = " << hexd(0.5 * P.dt) << ", QDT2 = " << hexd(0.25 * P.dt2)
      << ", STT_S = " << hexd(P.stt_s) << ", STT_X = " << hexd(P.stt_x) << ";\n";
    o << "}  // namespace specc\nnamespace spec {\n";
    TmaGeo gp, gc;
    std::string why;
    const bool tma = plan_tma(s, gp, gc, why);
    if (tma) { emit_tma_geo(o, "TmaP", gp); emit_tma_geo(o, "TmaC", gc); }
    o << "}  // namespace spec\n";
    int fg[4];
    size_t fsmem = 0;
    if (plan_fused(s, fg, fsmem))
        o << "namespace spec { constexpr int FTX = " << fg[0] << ", FTY = " << fg[1] << ", FTZ = " << fg[2] << ", FNT = " << fg[3] << "; }\n#define SPIN_FUSED 1\n";
    int cg[4];
    const bool col = plan_col(s, cg);
    if (col) o << "namespace spec { constexpr int CBX = " << cg[0] << ", CBY = " << cg[1] << ", CCZ = " << cg[2] << ", CNZC = " << cg[3] << "; }\n#define SPIN_COL 1\n";
    int pg[3];
    if (plan_pair(s, pg)) o << "namespace spec { constexpr int VBX = " << pg[0] << ", VBY = " << pg[1] << ", VBZ = " << pg[2] << "; }\n#define SPIN_PAIR 1\n";
    if (tma) o << "#define SPIN_TMA 1\n";
    o << "#include \"spin_jit_kernels.cuh\"\n";
    return o.str();
}

// compile `source` for sm_100a; on success the cubin is returned in `cubin`
// process-wide cache of compiled translation units: systems with the same plan (replicas, option toggles that do not change the
// source, test fixtures) share one NVRTC compilation
namespace {
std::mutex g_cache_mutex;
std::map<std::string, std::string> g_cubin_cache;
}

// NVRTC is bound at run time, by PATH: a process that imported torch has torch's own libnvrtc.so.12 (12.8) loaded under the same
// soname, and a link-time dependency would silently resolve to it.  The toolkit's 12.9 (the one nvcc built this library with) keeps the
// corrector at 40 registers where 12.8 needs 48 (6 instead of 5 blocks per SM, 4 % of the cfg3 step).  Order: $SPINLLG_NVRTC, the
// toolkit the library was built with (SPIN_NVRTC_PATH, set by build.py), then whatever the loader finds under the soname.
namespace {
struct Nvrtc {
    decltype(&nvrtcCreateProgram) CreateProgram;
    decltype(&nvrtcCompileProgram) CompileProgram;
    decltype(&nvrtcGetProgramLogSize) GetProgramLogSize;
    decltype(&nvrtcGetProgramLog) GetProgramLog;
    decltype(&nvrtcGetCUBINSize) GetCUBINSize;
    decltype(&nvrtcGetCUBIN) GetCUBIN;
    decltype(&nvrtcDestroyProgram) DestroyProgram;
    decltype(&nvrtcGetErrorString) GetErrorString;
    decltype(&nvrtcVersion) Version;
    std::string path;
    bool ok;
};
const Nvrtc &nvrtc() {
    static const Nvrtc api = [] {
        Nvrtc a;
        memset((void *)&a, 0, offsetof(Nvrtc, path));
        a.ok = false;
        std::vector<std::string> cands;
        if (const char *e = getenv("SPINLLG_NVRTC")) cands.push_back(e);
#ifdef SPIN_NVRTC_PATH
        cands.push_back(SPIN_NVRTC_PATH);
#endif
        cands.push_back("libnvrtc.so.12");
        cands.push_back("libnvrtc.so");
        for (const std::string &c : cands) {
            void *h = dlopen(c.c_str(), RTLD_NOW | RTLD_LOCAL);
            if (!h) continue;
#define SPIN_NVRTC_SYM(f) a.f = (decltype(a.f))dlsym(h, "nvrtc" #f)
            SPIN_NVRTC_SYM(CreateProgram); SPIN_NVRTC_SYM(CompileProgram); SPIN_NVRTC_SYM(GetProgramLogSize); SPIN_NVRTC_SYM(GetProgramLog);
            SPIN_NVRTC_SYM(GetCUBINSize); SPIN_NVRTC_SYM(GetCUBIN); SPIN_NVRTC_SYM(DestroyProgram); SPIN_NVRTC_SYM(GetErrorString);
            SPIN_NVRTC_SYM(Version);
#undef SPIN_NVRTC_SYM
            if (a.CreateProgram && a.CompileProgram && a.GetProgramLogSize && a.GetProgramLog && a.GetCUBINSize && a.GetCUBIN &&
                a.DestroyProgram && a.GetErrorString && a.Version) {
                // a trial compilation: an NVRTC that cannot find its builtins library loads fine and fails only here
                nvrtcProgram prog;
                bool works = false;
                if (a.CreateProgram(&prog, "extern \"C\" __global__ void spin_probe(double *x) { x[0] = 1.0; }\n", "spin_probe.cu", 0, nullptr,
                                    nullptr) == NVRTC_SUCCESS) {
                    const char *opts[] = {"--gpu-architecture=sm_100a"};
                    works = a.CompileProgram(prog, 1, opts) == NVRTC_SUCCESS;
                    a.DestroyProgram(&prog);
                }
                if (works) {
                    a.path = c;
                    a.ok = true;
                    break;
                }
            }
            dlclose(h);
        }
        return a;
    }();
    return api;
}
}  // namespace

static bool nvrtc_at_least(int major, int minor) {
    const Nvrtc &rt = nvrtc();
    int ma = 0, mi = 0;
    if (!rt.ok || rt.Version(&ma, &mi) != NVRTC_SUCCESS) return false;
    return ma > major || (ma == major && mi >= minor);
}

// "12.9 (/usr/local/cuda/lib64/libnvrtc.so.12)" or why there is none
std::string spin::jit_compiler_info() {
    const Nvrtc &rt = nvrtc();
    if (!rt.ok) return "NVRTC not found";
    int major = 0, minor = 0;
    rt.Version(&major, &minor);
    return std::to_string(major) + "." + std::to_string(minor) + " (" + rt.path + ")";
}

int spin::jit_compile(const std::string &source, std::string &cubin, std::string &log) {
    const Nvrtc &rt = nvrtc();
    if (!rt.ok) return spin::fail(SPIN_ERR_CUDA, "NVRTC (libnvrtc.so.12) could not be loaded");
    {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        auto it = g_cubin_cache.find(source);
        if (it != g_cubin_cache.end() && !getenv("SPINLLG_JIT_DUMP")) { cubin = it->second; log.clear(); return SPIN_OK; }
    }
    nvrtcProgram prog;
    if (rt.CreateProgram(&prog, source.c_str(), "spin_jit_spec.cu", 0, nullptr, nullptr) != NVRTC_SUCCESS)
        return spin::fail(SPIN_ERR_CUDA, "nvrtcCreateProgram failed");
    const std::string inc = "-I" + csrc_dir();
    const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "-default-device", inc.c_str()};
    const nvrtcResult r = rt.CompileProgram(prog, 5, opts);
    size_t n = 0;
    rt.GetProgramLogSize(prog, &n);
    log.assign(n, '\0');
    if (n) rt.GetProgramLog(prog, &log[0]);
    if (r != NVRTC_SUCCESS) {
        rt.DestroyProgram(&prog);
        return spin::fail(SPIN_ERR_CUDA, "NVRTC compilation failed: %s | %.300s", rt.GetErrorString(r), log.c_str());
    }
    size_t nc = 0;
    rt.GetCUBINSize(prog, &nc);
    cubin.assign(nc, '\0');
    rt.GetCUBIN(prog, &cubin[0]);
    rt.DestroyProgram(&prog);
    {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        if (g_cubin_cache.size() >= 64) g_cubin_cache.clear();
        g_cubin_cache[source] = cubin;
    }
    if (const char *dump = getenv("SPINLLG_JIT_DUMP")) {       // developer aid: <dump>.cu / <dump>.cubin for cuobjdump -sass
        const std::string base(dump);
        if (FILE *f = fopen((base + ".cu").c_str(), "w")) { fwrite(source.data(), 1, source.size(), f); fclose(f); }
        if (FILE *f = fopen((base + ".cubin").c_str(), "wb")) { fwrite(cubin.data(), 1, cubin.size(), f); fclose(f); }
    }
    return SPIN_OK;
}

void spin::jit_release(spin_system *s) {
    JitState *j = s->jit;
    if (!j) return;
    if (j->loaded) cudaLibraryUnload(j->lib);
    delete j;
    s->jit = nullptr;
}

// CUtensorMap of one per-spin array: dims (x: PA, comp: 3, y: PB, z: PC, sublattice: nb), box = one staged plane
static int encode_plane_map(const spin_system *s, const TmaGeo &g, const double *base, CUtensorMap *tm) {
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn || qr != cudaDriverEntryPointSuccess)
            return spin::fail(SPIN_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
        encode = (encode_fn)fn;
    }
    const DevicePlan &P = s->plan;
    const cuuint64_t dims[5] = {(cuuint64_t)P.PA, 3, (cuuint64_t)P.PB, (cuuint64_t)P.PC, (cuuint64_t)P.nb};
    const cuuint64_t strides[4] = {(cuuint64_t)P.PA * 8, (cuuint64_t)3 * P.PA * 8, (cuuint64_t)3 * P.PA * P.PB * 8, (cuuint64_t)P.sub * 8};
    const cuuint32_t box[5] = {(cuuint32_t)(g.tbx + 2 * ((P.rA + 1) / 2 * 2)), 3, (cuuint32_t)(g.tby + 2 * P.rB), 1, (cuuint32_t)P.nb};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return spin::fail(SPIN_ERR_CUDA, "cuTensorMapEncodeTiled failed with code %d", (int)r);
    return SPIN_OK;
}

// kernels, launch geometry and tensor maps of the TMA-fed sweeps; on failure j->tma stays false and j->tma_note says why
static void tma_prepare(spin_system *s, JitState *j) {
    j->tma = false;
    if (!plan_tma(s, j->gp, j->gc, j->tma_note)) return;
    cudaError_t e = cudaLibraryGetKernel(&j->k_pred_tma, j->lib, "jit_predictor_tma");
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->k_corr_tma, j->lib, "jit_corrector_tma");
    if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)j->k_pred_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j->gp.smem_bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)j->k_corr_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j->gc.smem_bytes);
    int occ_p = 0, occ_c = 0;
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_p, (const void *)j->k_pred_tma, j->gp.tbx * j->gp.tby * j->gp.kz, j->gp.smem_bytes);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_c, (const void *)j->k_corr_tma, j->gc.tbx * j->gc.tby * j->gc.kz, j->gc.smem_bytes);
    if (e != cudaSuccess) { cudaGetLastError(); j->tma_note = std::string("TMA kernel setup failed: ") + cudaGetErrorString(e); return; }
    if (occ_p < 1 || occ_c < 1) { j->tma_note = "TMA kernels do not fit on an SM"; return; }
    const int sms = sm_count(s);
    j->grid_p = std::min(j->gp.items, sms * occ_p);
    j->grid_c = std::min(j->gc.items, sms * occ_c);
    if (encode_plane_map(s, j->gp, s->d_n[0], &j->tm_n[0]) || encode_plane_map(s, j->gp, s->d_n[1], &j->tm_n[1]) ||
        encode_plane_map(s, j->gc, s->d_n[0], &j->tm_cn[0]) || encode_plane_map(s, j->gc, s->d_n[1], &j->tm_cn[1]) ||
        encode_plane_map(s, j->gc, s->d_np, &j->tm_cnp)) { j->tma_note = spin_last_error(); return; }
    j->tma = true;
    j->tma_note.clear();
}

// which variants of the sweeps this system can use (depends on options, solver, pins, image count -- not only on the source)
static void variants_prepare(spin_system *s, JitState *j) {
    tma_prepare(s, j);
    j->fused = plan_fused(s, j->fused_geo, j->fused_smem);
    if (j->fused) {
        cudaError_t fe = cudaLibraryGetKernel(&j->k_fused, j->lib, "jit_depondt_fused");
        if (fe == cudaSuccess) fe = cudaFuncSetAttribute((const void *)j->k_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j->fused_smem);
        if (fe != cudaSuccess) { cudaGetLastError(); j->fused = false; }
    }
    j->coop = false;
    j->cluster = false;
    if (s->opt_coop && !s->ddi_on && s->solver != SPIN_SOLVER_RK4 && s->n_img == 1) {
        int dev = 0, can = 0, occ = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&can, cudaDevAttrCooperativeLaunch, dev);
        dim3 grid, block;
        jit_brick_launch(s, grid, block);
        cudaError_t ce = cudaLibraryGetKernel(&j->k_coop, j->lib, "jit_steps_coop");
        if (ce == cudaSuccess) ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)j->k_coop, (int)block.x, 0);
        if (ce == cudaSuccess && can && occ > 0) {
            j->coop_grid = std::min((int)(grid.x * grid.y), occ * sm_count(s));
            j->coop = true;
        } else {
            cudaGetLastError();
        }
        // one cluster for the whole lattice: up to 8 blocks is portable, up to 16 needs the non-portable opt-in
        j->cluster = false;
        const int items = (int)(grid.x * grid.y);
        if (j->coop && s->opt_coop != 3 && items <= 16) {
            cudaError_t ke = cudaLibraryGetKernel(&j->k_cluster, j->lib, "jit_steps_cluster");
            if (ke == cudaSuccess && items > 8) ke = cudaFuncSetAttribute((const void *)j->k_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (ke == cudaSuccess) {
                cudaLaunchConfig_t cfg;
                memset(&cfg, 0, sizeof(cfg));
                cfg.gridDim = dim3((unsigned)items); cfg.blockDim = block;
                cudaLaunchAttribute at;
                at.id = cudaLaunchAttributeClusterDimension;
                at.val.clusterDim.x = (unsigned)items; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
                cfg.attrs = &at; cfg.numAttrs = 1;
                int nclusters = 0;
                ke = cudaOccupancyMaxActiveClusters(&nclusters, (const void *)j->k_cluster, &cfg);
                if (ke == cudaSuccess && nclusters >= 1) j->cluster = true;
            }
            if (ke != cudaSuccess) cudaGetLastError();
        }
    }
    j->col = plan_col(s, j->col_geo);
    if (j->col) {
        cudaError_t e = cudaLibraryGetKernel(&j->k_pred_col, j->lib, "jit_predictor_col");
        if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->k_corr_col, j->lib, "jit_corrector_col");
        if (e != cudaSuccess) { cudaGetLastError(); j->col = false; }
    }
    j->pair = plan_pair(s, j->pair_geo);
    if (j->pair) {
        cudaError_t e = cudaLibraryGetKernel(&j->k_pred_pair, j->lib, "jit_predictor_pair");
        if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->k_corr_pair, j->lib, "jit_corrector_pair");
        if (e != cudaSuccess) { cudaGetLastError(); j->pair = false; }
    }
}

int spin::jit_prepare(spin_system *s) {
    const std::string src = jit_source(s);
    if (s->jit && s->jit->loaded && s->jit->source == src) {      // plan changed in ways the sweeps do not see
        variants_prepare(s, s->jit);                              // the arrays may have moved, options may have changed
        return SPIN_OK;
    }
    jit_release(s);
    JitState *j = new JitState();
    j->loaded = false;
    j->tma = false;
    j->col = false;
    j->pair = false;
    j->coop = false;
    j->fused = false;
    j->source = src;
    s->jit = j;
    std::string cubin;
    int rc = jit_compile(src, cubin, j->log);
    if (rc) return rc;
    cudaError_t e = cudaLibraryLoadData(&j->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e != cudaSuccess) return spin::fail(SPIN_ERR_CUDA, "cudaLibraryLoadData failed: %s", cudaGetErrorString(e));
    j->loaded = true;
    e = cudaLibraryGetKernel(&j->k_pred, j->lib, "jit_predictor");
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->k_corr, j->lib, "jit_corrector");
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->k_rk4, j->lib, "jit_rk4_stage");
    if (e != cudaSuccess) return spin::fail(SPIN_ERR_CUDA, "cudaLibraryGetKernel failed: %s", cudaGetErrorString(e));
    variants_prepare(s, j);
    return SPIN_OK;
}

bool spin::jit_ready(const spin_system *s) { return s->jit && s->jit->loaded; }

// a brick sweep, launched with programmatic stream serialisation when the kernels were generated with spec::PDL (they then execute
// griddepcontrol.wait before their first dependent access): the blocks of the sweep become resident while the previous kernel drains
static cudaError_t launch_sweep(const spin_system *s, cudaKernel_t k, dim3 grid, dim3 block, void **args) {
    if (!pdl_mode(s)) return cudaLaunchKernel((const void *)k, grid, block, args, 0, s->stream);
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.stream = s->stream;
    cudaLaunchAttribute at;
    memset(&at, 0, sizeof(at));
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &at; cfg.numAttrs = 1;
    return cudaLaunchKernelExC(&cfg, (const void *)k, args);
}

int spin::jit_launch_predictor(spin_system *s, dim3 grid, dim3 block, const double *n, const double *fddi, double *np, double *Aout,
                               unsigned step_add) {
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    const unsigned char *pin = s->d_pin;
    const double *img_sigma = s->d_img_sigma;
    void *args[] = {(void *)&n, (void *)&fddi, (void *)&np, (void *)&Aout, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi,
                    (void *)&pin, (void *)&img_sigma};
    jit_brick_launch(s, grid, block);
    grid.z = (unsigned)s->n_img;
    SPIN_CUDA(launch_sweep(s, s->jit->k_pred, grid, block, args));
    return SPIN_OK;
}

int spin::jit_launch_corrector(spin_system *s, dim3 grid, dim3 block, const double *n, const double *np, const double *fddi_n,
                               const double *fddi_np, const double *Ain, double *nout, unsigned step_add) {
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned char *pin = s->d_pin;
    const double *img_sigma = s->d_img_sigma;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&n, (void *)&np, (void *)&fddi_n, (void *)&fddi_np, (void *)&Ain, (void *)&nout, (void *)&d_step, (void *)&step_add,
                    (void *)&seed_lo, (void *)&seed_hi, (void *)&pin, (void *)&img_sigma};
    jit_brick_launch(s, grid, block);
    grid.z = (unsigned)s->n_img;
    SPIN_CUDA(launch_sweep(s, s->jit->k_corr, grid, block, args));
    return SPIN_OK;
}

int spin::jit_launch_rk4_stage(spin_system *s, const double *base, const double *y, double *ynext, double *acc, double *noise,
                                const double *fddi, int stage, unsigned step_add) {
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    const unsigned char *pin = s->d_pin;
    void *args[] = {(void *)&base, (void *)&y, (void *)&ynext, (void *)&acc, (void *)&noise, (void *)&fddi, (void *)&stage, (void *)&d_step,
                    (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi, (void *)&pin};
    dim3 grid, block;
    jit_brick_launch(s, grid, block);
    SPIN_CUDA(cudaLaunchKernel((const void *)s->jit->k_rk4, grid, block, args, 0, s->stream));
    return SPIN_OK;
}

bool spin::jit_fused_ready(const spin_system *s) { return s->jit && s->jit->loaded && s->jit->fused; }

int spin::jit_launch_fused(spin_system *s, const double *n, double *nout, unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    const unsigned char *pin = s->d_pin;
    void *args[] = {(void *)&n, (void *)&nout, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi, (void *)&pin};
    const int *g = j->fused_geo;
    const unsigned tiles = (unsigned)(((s->nc[0] + g[0] - 1) / g[0]) * ((s->nc[1] + g[1] - 1) / g[1]) * ((s->nc[2] + g[2] - 1) / g[2]));
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_fused, dim3(tiles), dim3((unsigned)g[3]), args, j->fused_smem, s->stream));
    return SPIN_OK;
}

bool spin::jit_coop_ready(const spin_system *s) { return s->jit && s->jit->loaded && s->jit->coop; }
bool spin::jit_cluster_ready(const spin_system *s) { return jit_coop_ready(s) && s->jit->cluster; }

// nsteps Depondt/Heun/SIB steps in one cooperative launch; reads n from d_n[cur], leaves the result in d_n[cur ^ (nsteps & 1)]
int spin::jit_launch_steps_coop(spin_system *s, unsigned nsteps) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    double *n0 = s->d_n[s->cur], *n1 = s->d_n[s->cur ^ 1], *np = s->d_np, *aux = s->d_A;
    const unsigned char *pin = s->d_pin;
    unsigned int *bar = s->d_bar;
    dim3 grid, block;
    jit_brick_launch(s, grid, block);
    if (j->cluster) {
        void *cargs[] = {(void *)&n0, (void *)&n1, (void *)&np, (void *)&aux, (void *)&d_step, (void *)&nsteps, (void *)&seed_lo, (void *)&seed_hi, (void *)&pin};
        const unsigned items = grid.x * grid.y;
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(items); cfg.blockDim = block; cfg.stream = s->stream;
        cudaLaunchAttribute at;
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = items; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
        cfg.attrs = &at; cfg.numAttrs = 1;
        SPIN_CUDA(cudaLaunchKernelExC(&cfg, (const void *)j->k_cluster, cargs));
        return SPIN_OK;
    }
    SPIN_CUDA(cudaMemsetAsync(bar, 0, sizeof(unsigned int), s->stream));
    void *args[] = {(void *)&n0, (void *)&n1, (void *)&np, (void *)&aux, (void *)&d_step, (void *)&nsteps, (void *)&seed_lo, (void *)&seed_hi,
                    (void *)&pin, (void *)&bar};
    SPIN_CUDA(cudaLaunchCooperativeKernel((const void *)j->k_coop, dim3((unsigned)j->coop_grid), block, args, 0, s->stream));
    return SPIN_OK;
}

bool spin::jit_col_ready(const spin_system *s) { return s->jit && s->jit->loaded && s->jit->col; }

static void col_launch_dims(const spin_system *s, const JitState *j, dim3 &grid, dim3 &block) {
    const int *g = j->col_geo;
    grid = dim3((unsigned)(((s->nc[0] + g[0] - 1) / g[0]) * ((s->nc[1] + g[1] - 1) / g[1]) * g[3]), (unsigned)s->nb, 1);
    block = dim3((unsigned)(g[0] * g[1]), 1, 1);
}

int spin::jit_launch_predictor_col(spin_system *s, const double *n, const double *fddi, double *np, unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&n, (void *)&fddi, (void *)&np, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi};
    dim3 grid, block;
    col_launch_dims(s, j, grid, block);
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_pred_col, grid, block, args, 0, s->stream));
    return SPIN_OK;
}

int spin::jit_launch_corrector_col(spin_system *s, const double *n, const double *np, const double *fddi_n, const double *fddi_np, double *nout,
                                   unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&n, (void *)&np, (void *)&fddi_n, (void *)&fddi_np, (void *)&nout, (void *)&d_step, (void *)&step_add, (void *)&seed_lo,
                    (void *)&seed_hi};
    dim3 grid, block;
    col_launch_dims(s, j, grid, block);
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_corr_col, grid, block, args, 0, s->stream));
    return SPIN_OK;
}

bool spin::jit_pair_ready(const spin_system *s) { return s->jit && s->jit->loaded && s->jit->pair; }

static void pair_launch_dims(const spin_system *s, const JitState *j, dim3 &grid, dim3 &block) {
    const int *g = j->pair_geo;
    grid = dim3((unsigned)(((s->nc[0] + g[0] - 1) / g[0]) * ((s->nc[1] + g[1] - 1) / g[1]) * ((s->nc[2] + g[2] - 1) / g[2])), (unsigned)s->nb, 1);
    block = dim3((unsigned)(g[0] / 2 * g[1] * g[2]), 1, 1);
}

int spin::jit_launch_predictor_pair(spin_system *s, const double *n, const double *fddi, double *np, unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&n, (void *)&fddi, (void *)&np, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi};
    dim3 grid, block;
    pair_launch_dims(s, j, grid, block);
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_pred_pair, grid, block, args, 0, s->stream));
    return SPIN_OK;
}

int spin::jit_launch_corrector_pair(spin_system *s, const double *n, const double *np, const double *fddi_n, const double *fddi_np, double *nout,
                                    unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&n, (void *)&np, (void *)&fddi_n, (void *)&fddi_np, (void *)&nout, (void *)&d_step, (void *)&step_add, (void *)&seed_lo,
                    (void *)&seed_hi};
    dim3 grid, block;
    pair_launch_dims(s, j, grid, block);
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_corr_pair, grid, block, args, 0, s->stream));
    return SPIN_OK;
}

bool spin::jit_tma_ready(const spin_system *s) { return s->jit && s->jit->loaded && s->jit->tma; }
const char *spin::jit_tma_note(const spin_system *s) { return s->jit ? s->jit->tma_note.c_str() : "specialised kernels not loaded"; }

// the corrector stages n and n^p with its own tile: the maps are encoded per sweep geometry
int spin::jit_launch_predictor_tma(spin_system *s, int cur, const double *fddi, double *np, unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&j->tm_n[cur], (void *)&fddi, (void *)&np, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi};
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_pred_tma, dim3((unsigned)j->grid_p), dim3((unsigned)(j->gp.tbx * j->gp.tby * j->gp.kz)), args, j->gp.smem_bytes, s->stream));
    return SPIN_OK;
}

int spin::jit_launch_corrector_tma(spin_system *s, int cur, const double *fddi_n, const double *fddi_np, double *nout, unsigned step_add) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&j->tm_cn[cur], (void *)&j->tm_cnp, (void *)&fddi_n, (void *)&fddi_np, (void *)&nout, (void *)&d_step, (void *)&step_add,
                    (void *)&seed_lo, (void *)&seed_hi};
    SPIN_CUDA(cudaLaunchKernel((const void *)j->k_corr_tma, dim3((unsigned)j->grid_c), dim3((unsigned)(j->gc.tbx * j->gc.tby * j->gc.kz)), args, j->gc.smem_bytes, s->stream));
    return SPIN_OK;
}

const char *spin::jit_log(const spin_system *s) { return s->jit ? s->jit->log.c_str() : ""; }
