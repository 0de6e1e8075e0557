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

struct JitState {
    cudaLibrary_t lib;
    cudaKernel_t k_pred, k_corr, k_rk4;
    bool loaded;
    std::string source, log;
    // the whole Depondt step in one pass (spin_jit_march.cuh)
    bool march;
    cudaKernel_t k_march;
    int march_ty, march_nzc, march_threads, march_items;
    size_t march_smem;
    CUtensorMap tm_march[2][SPIN_MAX_BASIS];      // n[0], n[1], per sublattice, with the staged plane of the kernel as box (the kernel takes nb of them)
    // all steps in one cooperative launch (launch-bound lattices)
    bool coop;
    cudaKernel_t k_coop;
    int coop_grid;
    bool cluster;             // the whole lattice is one thread-block cluster (<= 16 bricks): hardware barrier instead of the grid barrier
    cudaKernel_t k_cluster;
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

}  // namespace

// brick of the specialised brick kernels: BX x BY x BZ sites per block.  32 x 4 x 2 (flat lattices 32 x 8 x 1) was the fastest of the
// shapes measured on B200 (profiles/r1c_README.md, profiles/r2_README.md: 32x2x2, 32x4x1, 64x2x1, 32x2x4, 32x8x2, ... are 0.5-18 % slower)
static void jit_brick(const spin_system *s, int b[3]) {
    const bool flat = s->nc[2] < 2;
    b[0] = 32; b[1] = 4; b[2] = flat ? 1 : 2;
    // flat lattices: bricks of 32 x 4 (128 threads) spread a sweep over more SMs than 32 x 8 did (cfg4 35.8 -> 33.6, cfg1 3.39 -> 3.13 us
    // per step, cfg2 unchanged; 32 x 2: 33.8 / 3.25 / 15.1); 32 x 8 is kept where only that fits the one-cluster kernel (16 blocks)
    if (flat) {
        const int nbx = (s->nc[0] + 31) / 32;
        const long items4 = (long)nbx * ((s->nc[1] + 3) / 4) * s->nb, items8 = (long)nbx * ((s->nc[1] + 7) / 8) * s->nb;
        if (items4 > 16 && items8 <= 16) b[1] = 8;
    }
}
static void jit_brick_launch(const spin_system *s, dim3 &grid, dim3 &block);
// programmatic dependent launch of the brick sweeps: 0 off, 1 dependents released at entry, 2 at the end of each block.
// Measured (profiles/r1g_README.md): sweeps of many waves gain 1-3 % from 1 and lose with 2.  Sweeps of about one wave lose with 1 (the
// next sweep's blocks are placed while this one's still hold their SMs, unevenly); with 2 they gain 10-14 % when the kernels were
// compiled by NVRTC 12.9 and lose 4 % with NVRTC 12.8, so the automatic choice depends on the compiler that was found.
static bool nvrtc_at_least(int major, int minor);
static int pdl_mode(const spin_system *s) {
    if (s->slab_on) return 0;      // the sweeps of a slab also depend on halo copies made on another stream: plain stream order only
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

// geometry of the one-pass plane-marching kernel: rows per tile, chunks along c, threads, shared memory; false if it does not apply
namespace {
struct MarchGeo { int ra, rb, rc, ty, nzc, look, blocks, threads, items; size_t smem; };
bool plan_march(const spin_system *s, MarchGeo &g) {
    const DevicePlan &P = s->plan;
    if (!spin::march_eligible(s) || P.ghost_mult != 2) return false;
    g.ra = P.rA / 2; g.rb = P.rB / 2; g.rc = P.rC / 2;
    const bool flat = P.Nc == 1;      // one plane: nothing to march along, the kernel is "predictor of tile + rim, corrector of the tile"
    if ((g.rc < 1 && !flat) || g.ra > 4 || g.rb > 4 || g.rc > 2) return false;
    // flat lattices: one launch instead of two always pays while the step is latency-bound (cfg2 Hamiltonian, reach 2, thermal field:
    // 96^2 .. 256^2 sites 7.3-7.4 us against 8.2-9.3); at 512^2 the rim of two reaches (1.41 x the predictor work) loses to the brick
    // sweeps (25.4 against 21.6 us), with a reach of one it does not (cfg1 Hamiltonian: 7.9 against 8.6; 1024^2: 23.3 / 23.5)
    if (flat && s->opt_march < 2 && s->N > 131072 && std::max(g.ra, g.rb) > 1) return false;
    const int hx = (2 * g.ra + 1) / 2 * 2;
    if (P.LA < hx) return false;
    const int sms = sm_count(s);
    double best = -1.0;
    bool found = false;
    for (int look : {2, 3, 1})
    for (int ty : {8, 12, 16, 6, 4}) {                       // tile rows; prefer tiles that divide the lattice
        const int py = ty + 2 * g.rb, rimw = (2 * g.ra * py + 31) / 32, threads = 32 * (py + rimw);
        if (threads > 1024) continue;
        const size_t nslot = ((size_t)3 * (32 + 2 * hx) * (ty + 4 * g.rb) + 15) / 16 * 16, ppl = (size_t)3 * (32 + 2 * g.ra) * py;
        const size_t smem = ((size_t)(2 * g.rc + 1 + look) * nslot + (size_t)(2 * g.rc + 2) * ppl) * 8 * (size_t)s->nb + (size_t)(2 * g.rc + 1 + look) * 8;
        if (smem > 200 * 1024) continue;
        const int per_sm = (int)std::min<size_t>((size_t)(227 * 1024) / (smem + 1024), (size_t)std::min(2048 / threads, 65536 / (threads * 56)));
        if (per_sm < 1) continue;
        const int cols = ((P.Na + 31) / 32) * ((P.Nb + ty - 1) / ty), slots = sms * per_sm;
        for (int nzc = 1; nzc <= (flat ? 1 : P.Nc / 4); ++nzc) {
            const long items = (long)cols * nzc;
            const long waves = (items + slots - 1) / slots;
            const double cz = (double)P.Nc / nzc;
            // useful fraction: full waves x chunk overlap of the predictor x rim of the tile x rows that hang over the lattice
            // (one block per SM stalls the whole SM at its barrier, and one plane of look-ahead does not cover the HBM latency: measured 7 % and
            // 12-20 % slower on cfg3, profiles/r2_README.md)
            const double eff = (double)items / (double)(waves * slots) * cz / (cz + 2.0 * g.rc) * (32.0 * ty) / (double)((32 + 2 * g.ra) * py) *
                               (double)P.Nb / (double)(((P.Nb + ty - 1) / ty) * ty) * (per_sm == 1 ? 0.85 : 1.0) * (look == 1 ? 0.8 : (look == 3 ? 0.99 : 1.0));
            if (eff > best + 1e-9) { best = eff; found = true; g.ty = ty; g.nzc = nzc; g.look = look; g.blocks = per_sm; g.threads = threads; g.items = (int)items; g.smem = smem; }
        }
    }
    return found;
}
}  // namespace

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
    // corrector: the fields of n and of n^p one after the other (40 registers, 1.5 % faster on cfg3 than interleaved, 48 registers)
    o << "constexpr bool SPLIT_CORR = true;\n";
    // corrector bricks in reverse order (L2 reuse of what the predictor touched last): 68.1 -> 65.3 us per step on cfg3
    o << "constexpr bool REVERSE_CORR = true;\n";
    // programmatic dependent launch: the sweeps release their dependents at once and wait for their prerequisites in the kernel
    o << "constexpr int PDL = " << pdl_mode(s) << ";      // 0 off, 1 dependents released at entry, 2 at the end of the block\n";
    o << "constexpr bool MULTI_IMAGE = " << (s->n_img > 1 ? "true" : "false") << ";\n";
    o << "constexpr bool DAMPING_ONLY = " << (s->damping_only ? "true" : "false") << ";\n";
    o << "constexpr bool HAS_PIN = " << (s->d_pin ? "true" : "false") << ";\n";
    o << "constexpr int CELL_OFF = " << P.cell_off << ";      // global index of local cell 0 (slab decomposition)\n";
    // slab decomposition: first plane of this slab in the whole lattice and the planes of the whole lattice (else 0 and NC)
    o << "constexpr int C_OFF = " << (s->slab_on ? s->slab_off : 0) << ", GNC = " << (s->slab_on ? s->slab_gnc : P.Nc) << ";\n";
    o << "constexpr bool SLAB = " << (s->slab_on ? "true" : "false") << ";\n";
    o << "constexpr bool HAS_SITE_MU = " << (s->d_mu_ratio ? "true" : "false") << ";      // per-site moments (PAPER.md:79)\n";
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
    o << "}  // namespace spec\n";
    MarchGeo mg;
    if (plan_march(s, mg))
        o << "namespace spec { constexpr int MRA = " << mg.ra << ", MRB = " << mg.rb << ", MRC = " << mg.rc << ", MTY = " << mg.ty << ", MNZC = " << mg.nzc
          << ", MLOOK = " << mg.look << ", MBLOCKS = " << mg.blocks << "; }\n#define SPIN_MARCH 1\n";
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

// which variants of the sweeps this system can use (depends on options, solver, pins, image count -- not only on the source)
// tensor map of one spin array for the marching kernel: dims (x: PA, comp: 3, y: PB, z: PC), box = one staged plane (tile + rim)
static int encode_march_map(const spin_system *s, const MarchGeo &g, const double *base, CUtensorMap *tm) {
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
    const int hx = (2 * g.ra + 1) / 2 * 2;
    const cuuint64_t dims[4] = {(cuuint64_t)P.PA, 3, (cuuint64_t)P.PB, (cuuint64_t)P.PC};
    const cuuint64_t strides[3] = {(cuuint64_t)P.PA * 8, (cuuint64_t)3 * P.PA * 8, (cuuint64_t)3 * P.PA * P.PB * 8};
    const cuuint32_t box[4] = {(cuuint32_t)(32 + 2 * hx), 3, (cuuint32_t)(g.ty + 4 * g.rb), 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return spin::fail(SPIN_ERR_CUDA, "cuTensorMapEncodeTiled failed with code %d", (int)r);
    return SPIN_OK;
}

static void variants_prepare(spin_system *s, JitState *j) {
    j->march = false;
    MarchGeo mg;
    if (plan_march(s, mg)) {
        cudaError_t e = cudaLibraryGetKernel(&j->k_march, j->lib, "jit_depondt_march");
        if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)j->k_march, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mg.smem);
        int occ = 0;
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)j->k_march, mg.threads, mg.smem);
        bool maps = e == cudaSuccess && occ >= 1;
        for (int a = 0; a < 2 && maps; ++a)
            for (int b = 0; b < s->nb && maps; ++b) maps = encode_march_map(s, mg, s->d_n[a] + (size_t)b * s->plan.sub, &j->tm_march[a][b]) == SPIN_OK;
        if (maps) {
            j->march = true;
            j->march_ty = mg.ty; j->march_nzc = mg.nzc; j->march_threads = mg.threads; j->march_items = mg.items; j->march_smem = mg.smem;
        } else {
            cudaGetLastError();
        }
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
    j->coop = false;
    j->march = false;
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

void spin::jit_brick_shape(const spin_system *s, int b[3]) { jit_brick(s, b); }

// brick0 / nbricks: a range of bricks (slab decomposition: boundary planes first, interior while the halos travel); 0 bricks = all
int spin::jit_launch_predictor(spin_system *s, dim3 grid, dim3 block, const double *n, const double *fddi, double *np, double *Aout,
                               unsigned step_add, unsigned brick0, unsigned nbricks) {
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    const unsigned char *pin = s->d_pin;
    const double *img_sigma = s->d_img_sigma, *mu_ratio = s->d_mu_ratio;
    void *args[] = {(void *)&n, (void *)&fddi, (void *)&np, (void *)&Aout, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi,
                    (void *)&pin, (void *)&img_sigma, (void *)&mu_ratio, (void *)&brick0};
    jit_brick_launch(s, grid, block);
    if (nbricks) grid.x = nbricks;
    grid.z = (unsigned)s->n_img;
    SPIN_CUDA(launch_sweep(s, s->jit->k_pred, grid, block, args));
    return SPIN_OK;
}

int spin::jit_launch_corrector(spin_system *s, dim3 grid, dim3 block, const double *n, const double *np, const double *fddi_n,
                               const double *fddi_np, const double *Ain, double *nout, unsigned step_add, unsigned brick0, unsigned nbricks) {
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned char *pin = s->d_pin;
    const double *img_sigma = s->d_img_sigma, *mu_ratio = s->d_mu_ratio;
    const unsigned long long *d_step = s->d_step;
    void *args[] = {(void *)&n, (void *)&np, (void *)&fddi_n, (void *)&fddi_np, (void *)&Ain, (void *)&nout, (void *)&d_step, (void *)&step_add,
                    (void *)&seed_lo, (void *)&seed_hi, (void *)&pin, (void *)&img_sigma, (void *)&mu_ratio, (void *)&brick0};
    jit_brick_launch(s, grid, block);
    if (nbricks) grid.x = nbricks;
    grid.z = (unsigned)s->n_img;
    SPIN_CUDA(launch_sweep(s, s->jit->k_corr, grid, block, args));
    return SPIN_OK;
}

int spin::jit_launch_rk4_stage(spin_system *s, const double *base, const double *y, double *ynext, double *acc, double *noise,
                                const double *fddi, int stage, unsigned step_add) {
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    const unsigned char *pin = s->d_pin;
    const double *mu_ratio = s->d_mu_ratio;
    void *args[] = {(void *)&base, (void *)&y, (void *)&ynext, (void *)&acc, (void *)&noise, (void *)&fddi, (void *)&stage, (void *)&d_step,
                    (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi, (void *)&pin, (void *)&mu_ratio};
    dim3 grid, block;
    jit_brick_launch(s, grid, block);
    SPIN_CUDA(cudaLaunchKernel((const void *)s->jit->k_rk4, grid, block, args, 0, s->stream));
    return SPIN_OK;
}

bool spin::jit_march_ready(const spin_system *s) { return s->jit && s->jit->loaded && s->jit->march; }

// one Depondt step in one pass: reads d_n[cur] through its tensor map, writes nout
// part 0: every item; 1: the first and the last chunk along c (the planes a neighbouring slab needs), two launches; 2: the chunks in between
// peer_lo / peer_hi (slabs only, may be null): the neighbours' next configurations, into whose ghost layers the kernel writes its boundary planes
int spin::jit_launch_march(spin_system *s, int cur, double *nout, unsigned step_add, int part, double *peer_lo, double *peer_hi, int peer_lo_nc) {
    JitState *j = s->jit;
    unsigned seed_lo = s->plan.seed_lo, seed_hi = s->plan.seed_hi;
    const unsigned long long *d_step = s->d_step;
    const unsigned char *pin = s->d_pin;
    const double *mu_ratio = s->d_mu_ratio;
    unsigned item0 = 0;
    void *args[] = {(void *)&j->tm_march[cur][0], (void *)&nout, (void *)&d_step, (void *)&step_add, (void *)&seed_lo, (void *)&seed_hi, (void *)&pin, (void *)&mu_ratio,
                    (void *)&item0, (void *)&peer_lo, (void *)&peer_hi, (void *)&peer_lo_nc};
    const unsigned items = (unsigned)j->march_items, cols = items / (unsigned)j->march_nzc;      // items = chunk x column tile, chunk-major
    unsigned ranges[2][2] = {{0u, items}, {0u, 0u}};
    if (part == 1) { ranges[0][1] = cols; if (j->march_nzc > 1) { ranges[1][0] = items - cols; ranges[1][1] = items; } }
    else if (part == 2) { ranges[0][0] = cols; ranges[0][1] = j->march_nzc > 1 ? items - cols : cols; }
    for (int r = 0; r < 2; ++r) {
        if (ranges[r][1] <= ranges[r][0]) continue;
        item0 = ranges[r][0];
        SPIN_CUDA(cudaLaunchKernel((const void *)j->k_march, dim3(ranges[r][1] - ranges[r][0]), dim3((unsigned)j->march_threads), args, j->march_smem, s->stream));
        if (part) s->n_launch++;      // (part 0: counted by the caller)
    }
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
    const double *mu_ratio = s->d_mu_ratio;
    dim3 grid, block;
    jit_brick_launch(s, grid, block);
    if (j->cluster) {
        void *cargs[] = {(void *)&n0, (void *)&n1, (void *)&np, (void *)&aux, (void *)&d_step, (void *)&nsteps, (void *)&seed_lo, (void *)&seed_hi, (void *)&pin,
                         (void *)&mu_ratio};
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
                    (void *)&pin, (void *)&bar, (void *)&mu_ratio};
    SPIN_CUDA(cudaLaunchCooperativeKernel((const void *)j->k_coop, dim3((unsigned)j->coop_grid), block, args, 0, s->stream));
    return SPIN_OK;
}

const char *spin::jit_log(const spin_system *s) { return s->jit ? s->jit->log.c_str() : ""; }
