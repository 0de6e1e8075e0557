// spin_api.cu -- C-ABI entry points (include/spinllg.h), host planner and kernel launches.
//
// Host side of the path: geometry, the neighbour-shell finder, expansion of the unique pair / quadruplet lists into
// per-basis-atom gather tables (forward + backward entries, D sign flipped backward), LLG prefactors,
// and the launch sequence of one Depondt step (App. B :369-380):
//     [DDI(n)] -> predictor -> [DDI(n^p)] -> corrector          (2 own kernels per step without DDI)
// captured into a CUDA graph for launch-bound lattices.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <mutex>

#include "spin_kernels.cuh"

using namespace spin;

static int topo_noalloc_setup();      // resolves the device address of topological_charge_noalloc's scratch array (below)

// ---------------------------------------------------------------------------------------------- errors
static thread_local char g_err[512] = "";

int spin::fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
extern "C" const char *spin_last_error(void) { return g_err; }
extern "C" const char *spin_version(void) { return "spinllg-b200 0.1 (sm_100a, fp64)"; }

#define REQUIRE(cond, ...)                                   \
    do {                                                     \
        if (!(cond)) return spin::fail(SPIN_ERR_ARG, __VA_ARGS__); \
    } while (0)

static void drop_graphs(spin_system *s) {
    for (int k = 0; k < 2; ++k)
        if (s->graph_exec[k]) { cudaGraphExecDestroy(s->graph_exec[k]); s->graph_exec[k] = nullptr; }
    s->graph_steps = 0;
}

// ---------------------------------------------------------------------------------------------- brick shapes
// 2-D lattices use 32x8x1 bricks, 3-D lattices 32x4x2 (256 threads either way).
namespace {
struct Launch { dim3 grid, block; bool flat; };

Launch brick_launch(const spin_system *s) {
    Launch L;
    L.flat = s->nc[2] < 2;
    const int BX = 32, BY = L.flat ? 8 : 4, BZ = L.flat ? 1 : 2;
    const int nbx = (s->nc[0] + BX - 1) / BX, nby = (s->nc[1] + BY - 1) / BY, nbz = (s->nc[2] + BZ - 1) / BZ;
    L.grid = dim3((unsigned)(nbx * nby * nbz), (unsigned)s->nb, 1);
    L.block = dim3(256, 1, 1);
    return L;
}

void cart(const spin_system *s, const double f[3], double r[3]) {
    for (int k = 0; k < 3; ++k) r[k] = s->alat * (f[0] * s->brav[k] + f[1] * s->brav[3 + k] + f[2] * s->brav[6 + k]);
}

// translation reduced to the representative of smallest magnitude in a periodic direction
int reduce_translation(int t, int n, int periodic) {
    if (!periodic) return t;
    int r = t % n;
    if (r < 0) r += n;
    if (2 * r > n) r -= n;
    return r;
}

// ------------------------------------------------------------------------------------------ neighbour shells
// All bonds (bi -> bj at translation t) sorted by length and grouped into shells; each bond once (the partner
// direction (bj -> bi, -t) is the same bond).  Only directions with more than one cell are scanned.
struct Bond { int bi, bj, t[3]; double r[3], len; };

std::vector<std::vector<Bond>> find_shells(const spin_system *s, int n_shells) {
    std::vector<std::vector<Bond>> shells;
    for (int range = 2;; ++range) {
        std::vector<Bond> all;
        int lim[3];
        for (int d = 0; d < 3; ++d) lim[d] = (s->nc[d] > 1) ? range : 0;
        for (int bi = 0; bi < s->nb; ++bi)
            for (int bj = 0; bj < s->nb; ++bj)
                for (int t0 = -lim[0]; t0 <= lim[0]; ++t0)
                    for (int t1 = -lim[1]; t1 <= lim[1]; ++t1)
                        for (int t2 = -lim[2]; t2 <= lim[2]; ++t2) {
                            if (bi == bj && t0 == 0 && t1 == 0 && t2 == 0) continue;
                            // keep one representative of {(bi,bj,t), (bj,bi,-t)}
                            const int key_a[5] = {bi, bj, t0, t1, t2}, key_b[5] = {bj, bi, -t0, -t1, -t2};
                            if (std::lexicographical_compare(key_b, key_b + 5, key_a, key_a + 5)) continue;
                            Bond b;
                            b.bi = bi; b.bj = bj; b.t[0] = t0; b.t[1] = t1; b.t[2] = t2;
                            const double f[3] = {t0 + s->basis[3 * bj] - s->basis[3 * bi], t1 + s->basis[3 * bj + 1] - s->basis[3 * bi + 1],
                                                 t2 + s->basis[3 * bj + 2] - s->basis[3 * bi + 2]};
                            cart(s, f, b.r);
                            b.len = sqrt(b.r[0] * b.r[0] + b.r[1] * b.r[1] + b.r[2] * b.r[2]);
                            all.push_back(b);
                        }
        std::stable_sort(all.begin(), all.end(), [](const Bond &x, const Bond &y) { return x.len < y.len; });
        shells.clear();
        const double tol = 1e-6 * s->alat;
        for (const Bond &b : all) {
            if (shells.empty() || b.len > shells.back().front().len + tol) shells.emplace_back();
            shells.back().push_back(b);
        }
        // shells are complete only up to the radius the scan certainly covers
        double rmin = 1e300;
        for (int d = 0; d < 3; ++d) {
            if (lim[d] == 0) continue;
            // distance between lattice planes along direction d bounds what a scan of `range` cells covers
            double a[3], b2[3], c[3];
            const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
            for (int k = 0; k < 3; ++k) { a[k] = s->brav[3 * d + k]; b2[k] = s->brav[3 * d1 + k]; c[k] = s->brav[3 * d2 + k]; }
            double nrm[3] = {b2[1] * c[2] - b2[2] * c[1], b2[2] * c[0] - b2[0] * c[2], b2[0] * c[1] - b2[1] * c[0]};
            const double nn = sqrt(nrm[0] * nrm[0] + nrm[1] * nrm[1] + nrm[2] * nrm[2]);
            const double h = fabs(a[0] * nrm[0] + a[1] * nrm[1] + a[2] * nrm[2]) / nn * s->alat;
            rmin = std::min(rmin, h * (range - 1));
        }
        int complete = 0;
        for (auto &sh : shells) if (sh.front().len < rmin - tol) ++complete; else break;
        if (complete >= n_shells || range > 12 || rmin == 1e300) {
            shells.resize(std::min<size_t>(shells.size(), (size_t)n_shells));
            return shells;
        }
    }
}

// ------------------------------------------------------------------------------------------ plan
int stt_coefficients(const spin_system *s, double cd[3]) {
    // j^ = sum_d c_d a_d over the directions with more than one cell (least squares if fewer than three)
    int act[3], na = 0;
    for (int d = 0; d < 3; ++d) { cd[d] = 0.0; if (s->nc[d] > 1) act[na++] = d; }
    if (na == 0) return 0;
    double G[3][4];
    for (int p = 0; p < na; ++p) {
        double ap[3];
        for (int k = 0; k < 3; ++k) ap[k] = s->alat * s->brav[3 * act[p] + k];
        G[p][3] = ap[0] * s->jdir[0] + ap[1] * s->jdir[1] + ap[2] * s->jdir[2];
        for (int q = 0; q < na; ++q) {
            double aq[3];
            for (int k = 0; k < 3; ++k) aq[k] = s->alat * s->brav[3 * act[q] + k];
            G[p][q] = ap[0] * aq[0] + ap[1] * aq[1] + ap[2] * aq[2];
        }
    }
    for (int p = 0; p < na; ++p) {          // Gauss-Jordan with partial pivoting on the normal equations
        int piv = p;
        for (int r = p + 1; r < na; ++r) if (fabs(G[r][p]) > fabs(G[piv][p])) piv = r;
        if (fabs(G[piv][p]) < 1e-300) return -1;
        if (piv != p) for (int q = 0; q < 4; ++q) std::swap(G[p][q], G[piv][q]);
        for (int r = 0; r < na; ++r) {
            if (r == p) continue;
            const double f = G[r][p] / G[p][p];
            for (int q = p; q < na; ++q) G[r][q] -= f * G[p][q];
            G[r][3] -= f * G[p][3];
        }
    }
    for (int p = 0; p < na; ++p) cd[act[p]] = G[p][3] / G[p][p];
    return 0;
}

}  // namespace
// The one-pass plane-marching kernel (spin_jit_march.cuh) applies to 3-D lattices of one basis atom advanced by the Depondt or the Heun
// solver (the two-stage explicit schemes: predictor from n, corrector from n and n^p) without dipolar coupling or images; lattices small enough for the all-steps-in-one-launch path keep that path.  A slab of a decomposed
// lattice takes it too (llg_slab_step: ONE halo exchange of depth 2 x reach per step instead of two of depth reach) unless it has pinned
// spins or per-site moments: the kernel recomputes the predictor of the neighbours' boundary planes and would need their flags.
bool spin::march_eligible(const spin_system *s) {
    if (s->slab_on && (s->d_pin || !s->mu_site.empty())) return false;
    // (several basis atoms, up to four: only on request, use_march = 2 -- measured on cfg4)
    const bool basis_ok = s->nb == 1 || (s->nb <= 4 && s->opt_march >= 2 && !s->slab_on);
    return s->opt_march && s->opt_jit && basis_ok && (s->solver == SPIN_SOLVER_DEPONDT || s->solver == SPIN_SOLVER_HEUN) && !s->ddi_on && s->n_img == 1 &&
           !s->opt_store_A &&
           s->nc[0] >= 32 && s->nc[1] >= 8 && (s->nc[2] >= 8 || s->nc[2] == 1) && (s->opt_march >= 2 || s->N >= (s->nc[2] == 1 ? 8192 : 65536));
}
namespace {
int build_plan(const spin_system *s, DevicePlan &P) {
    memset(&P, 0, sizeof(P));
    int reach[3] = {0, 0, 0};
    P.Na = s->nc[0]; P.Nb = s->nc[1]; P.Nc = s->nc[2];
    P.perA = s->per[0]; P.perB = s->per[1]; P.perC = s->per[2];
    P.nb = s->nb; P.Ncell = (int)s->ncell;
    const double a2 = 1.0 + s->alpha * s->alpha;
    for (int b = 0; b < s->nb; ++b) {
        const double m = s->mu[b] * MU_B;
        for (int k = 0; k < 3; ++k) P.zee[b][k] = m * s->Bmag * s->Bdir[k];
        P.pre[b] = -GAMMA / (a2 * m);
        P.sigma[b] = (s->T > 0.0) ? sqrt(2.0 * s->alpha * K_B * s->T * m / (GAMMA * s->dt_ps)) : 0.0;
        P.inv_mu[b] = 1.0 / m;
    }
    {   // anisotropy entries grouped by basis atom, list order kept within an atom
        int na = 0;
        for (int b = 0; b < s->nb; ++b) {
            P.ani_begin[b] = na;
            for (size_t e = 0; e < s->ani_b.size(); ++e) {
                if (s->ani_b[e] != b) continue;
                P.K2[na] = 2.0 * s->K[e];
                for (int k = 0; k < 3; ++k) P.Kax[na][k] = s->Kax[3 * e + k];
                ++na;
            }
        }
        P.ani_begin[s->nb] = na;
    }
    P.alpha = s->alpha; P.dt = s->dt_ps; P.dt2 = s->dt_ps * s->dt_ps;
    P.thermal_on = (s->T > 0.0) ? 1 : 0;
    P.seed_lo = (uint32_t)s->seed; P.seed_hi = (uint32_t)(s->seed >> 32);
    P.has_ddi = s->ddi_on ? 1 : 0;
    P.damping_only = s->damping_only;
    P.pin = s->d_pin;
    P.mu_ratio = s->d_mu_ratio;
    P.stt_on = (s->u != 0.0) ? 1 : 0;
    if (P.stt_on) {
        if (stt_coefficients(s, P.stt_c) != 0) return spin::fail(SPIN_ERR_ARG, "current direction: singular lattice metric");
        P.stt_s = -s->u * (s->alpha - s->beta) / a2;
        P.stt_x = s->u * (1.0 + s->alpha * s->beta) / a2;
        for (int d = 0; d < 3; ++d) if (P.stt_c[d] != 0.0) reach[d] = 1;
    }
    // ---- pair gather tables: every unique pair gives a forward entry for basis atom bi (+t, +D) and a backward
    // entry for bj (-t, -D).  Order per atom: all forward entries in list order, then all backward entries.
    std::vector<HostPair> all;
    all.insert(all.end(), s->pairs_explicit.begin(), s->pairs_explicit.end());
    all.insert(all.end(), s->pairs_exch_shells.begin(), s->pairs_exch_shells.end());
    all.insert(all.end(), s->pairs_dmi_shells.begin(), s->pairs_dmi_shells.end());
    // slab decomposition: translations along c are folded with the extent and boundary condition of the WHOLE lattice; the partner planes
    // outside this slab are its ghost layers, filled by the halo exchange
    const int Nd[3] = {s->nc[0], s->nc[1], s->slab_on ? s->slab_gnc : s->nc[2]};
    const int perd[3] = {s->per[0], s->per[1], s->slab_on ? s->slab_gper : s->per[2]};
    int ne = 0;
    for (int b = 0; b < s->nb; ++b) {
        P.pair_begin[b] = ne;
        for (int dir = 0; dir < 2; ++dir)
            for (const HostPair &p : all) {
                if ((dir == 0 ? p.bi : p.bj) != b) continue;
                const double sgn = dir == 0 ? 1.0 : -1.0;
                PairEntry e;
                memset(&e, 0, sizeof(e));
                int t[3];
                bool dead = false;
                for (int d = 0; d < 3; ++d) {
                    t[d] = reduce_translation((dir == 0 ? 1 : -1) * p.t[d], Nd[d], perd[d]);
                    if (!perd[d] && abs(t[d]) >= Nd[d]) dead = true;      // never inside an open lattice
                }
                if (dead) continue;
                e.da = t[0]; e.db = t[1]; e.dc = t[2];
                e.bj = dir == 0 ? p.bj : p.bi;
                e.J = p.J; e.Dx = sgn * p.D[0]; e.Dy = sgn * p.D[1]; e.Dz = sgn * p.D[2];
                // merge with an existing entry on the same partner (e.g. exchange shells + DMI shells on one bond)
                bool merged = false;
                for (int q = P.pair_begin[b]; q < ne; ++q) {
                    PairEntry &o = P.pairs[q];
                    if (o.bj == e.bj && o.da == e.da && o.db == e.db && o.dc == e.dc) {
                        o.J += e.J; o.Dx += e.Dx; o.Dy += e.Dy; o.Dz += e.Dz;
                        merged = true;
                        break;
                    }
                }
                if (merged) continue;
                if (ne >= SPIN_MAX_PAIR_ENTRIES)
                    return spin::fail(SPIN_ERR_LIMIT, "pair table needs more than %d gather entries", SPIN_MAX_PAIR_ENTRIES);
                P.pairs[ne++] = e;
                for (int d = 0; d < 3; ++d) reach[d] = std::max(reach[d], abs(t[d]));
            }
    }
    P.pair_begin[s->nb] = ne;
    // ---- quadruplet role tables (Eq. 2): role r of quadruplet q for basis atom b = q.b[r]
    int nq = 0;
    for (int b = 0; b < s->nb; ++b) {
        P.quad_begin[b] = nq;
        for (const HostQuad &q : s->quads) {
            int tm[4][3] = {{0, 0, 0}, {q.t[0], q.t[1], q.t[2]}, {q.t[3], q.t[4], q.t[5]}, {q.t[6], q.t[7], q.t[8]}};
            for (int role = 0; role < 4; ++role) {
                if (q.b[role] != b) continue;
                // F_role += K (n_Q . n_R) n_P
                const int Pm = role == 0 ? 1 : role == 1 ? 0 : role == 2 ? 3 : 2;
                const int Qm = role < 2 ? 2 : 0, Rm = role < 2 ? 3 : 1;
                const int mem[3] = {Pm, Qm, Rm};
                QuadEntry e;
                memset(&e, 0, sizeof(e));
                bool dead = false;
                for (int m = 0; m < 3; ++m) {
                    for (int d = 0; d < 3; ++d) {
                        const int t = reduce_translation(tm[mem[m]][d] - tm[role][d], Nd[d], perd[d]);
                        if (!perd[d] && abs(t) >= Nd[d]) dead = true;
                        e.d[m][d] = t;
                    }
                    e.b[m] = q.b[mem[m]];
                }
                if (dead) continue;      // some member can never be inside an open lattice
                for (int m = 0; m < 3; ++m) for (int d = 0; d < 3; ++d) reach[d] = std::max(reach[d], abs(e.d[m][d]));
                e.K = q.K;
                if (nq >= SPIN_MAX_QUAD_ENTRIES)
                    return spin::fail(SPIN_ERR_LIMIT, "quadruplet table needs more than %d role entries", SPIN_MAX_QUAD_ENTRIES);
                P.quads[nq++] = e;
            }
        }
    }
    P.quad_begin[s->nb] = nq;
    // ---- layout with ghost cells (spinllg_internal.h): ghost width = reach; rows start on 128-byte lines
    P.ghost_mult = march_eligible(s) ? 2 : 1;
    P.rA = P.ghost_mult * reach[0]; P.rB = P.ghost_mult * reach[1]; P.rC = P.ghost_mult * reach[2];
    P.gA = (P.perA && P.rA > 0) ? 1 : 0; P.gB = (P.perB && P.rB > 0) ? 1 : 0; P.gC = (P.perC && P.rC > 0 && !s->slab_on) ? 1 : 0;
    if (s->slab_on) {
        if (P.rC > P.Nc) return spin::fail(SPIN_ERR_ARG, "slab of %d planes is thinner than the reach %d of the Hamiltonian along c", P.Nc, P.rC);
        if (P.stt_on && P.stt_c[2] != 0.0) return spin::fail(SPIN_ERR_STATE, "slab decomposition needs an in-plane current (no component along c)");
        if (s->ddi_on) return spin::fail(SPIN_ERR_STATE, "the dipolar transform does not decompose into slabs (DESIGN.md section 8)");
        P.cell_off = s->slab_off * P.Na * P.Nb;
    }
    P.LA = (P.rA + 15) / 16 * 16; P.LB = P.rB; P.LC = P.rC;
    P.PA = P.LA + (P.Na + P.rA + 15) / 16 * 16; P.PB = P.Nb + 2 * P.rB; P.PC = P.Nc + 2 * P.rC;
    const int64_t sub = (int64_t)3 * P.PA * P.PB * P.PC;
    if (sub * s->nb >= (int64_t)2147483647) return spin::fail(SPIN_ERR_LIMIT, "padded lattice too large for 32-bit indexing");
    P.sub = (int)sub;
    auto lin = [&](int b, int bj, const int t[3]) { return (bj - b) * P.sub + (t[2] * P.PB + t[1]) * 3 * P.PA + t[0]; };
    for (int b = 0; b < s->nb; ++b) {
        for (int e = P.pair_begin[b]; e < P.pair_begin[b + 1]; ++e) {
            const int t[3] = {P.pairs[e].da, P.pairs[e].db, P.pairs[e].dc};
            P.pairs[e].lin = lin(b, P.pairs[e].bj, t);
        }
        for (int e = P.quad_begin[b]; e < P.quad_begin[b + 1]; ++e)
            for (int m = 0; m < 3; ++m) P.quads[e].lin[m] = lin(b, P.quads[e].b[m], P.quads[e].d[m]);
    }
    return SPIN_OK;
}

bool same_layout(const DevicePlan &a, const DevicePlan &b) {
    return a.LA == b.LA && a.LB == b.LB && a.LC == b.LC && a.PA == b.PA && a.PB == b.PB && a.PC == b.PC && a.sub == b.sub &&
           a.rA == b.rA && a.rB == b.rB && a.rC == b.rC && a.gA == b.gA && a.gB == b.gB && a.gC == b.gC;
}

#define NEED_DEVICE(s)                                                                                          \
    do {                                                                                                        \
        if (!(s)->has_device) return spin::fail(SPIN_ERR_CUDA, "no CUDA device: this library has no CPU fallback"); \
    } while (0)

// offset (in doubles) of the selected image in every per-spin array
inline size_t img_off(const spin_system *s) { return (size_t)s->img_sel * (size_t)s->nb * (size_t)s->plan.sub; }

// (re)allocate the per-spin arrays for the layout of `P`; the current configurations (all images) are carried over through a
// boundary-order staging buffer when `keep` is set
int allocate_arrays(spin_system *s, const DevicePlan &P, bool keep) {
    const int nt = 256;
    const unsigned nblk = (unsigned)((s->N + nt - 1) / nt);
    double *stage = s->d_aos;
    if (keep) {
        if (s->n_img > 1) SPIN_CUDA(cudaMalloc(&stage, (size_t)s->n_img * 3 * s->N * sizeof(double)));
        for (int k = 0; k < s->n_img; ++k)
            unpack_kernel<<<nblk, nt, 0, s->stream>>>(s->plan, s->d_n[s->cur] + (size_t)k * s->nb * s->plan.sub, stage + (size_t)k * 3 * s->N, (int)s->N, 0);
        s->n_launch += s->n_img;
        SPIN_CUDA(cudaStreamSynchronize(s->stream));
    }
    double **arrs[] = {&s->d_n[0], &s->d_n[1], &s->d_np, &s->d_A, &s->d_fddi[0], &s->d_fddi[1]};
    const size_t bytes = (size_t)s->n_img * s->nb * P.sub * sizeof(double);
    for (double **a : arrs) {
        if (*a) cudaFree(*a);
        *a = nullptr;
        cudaError_t e = cudaMalloc(a, bytes);
        if (e != cudaSuccess) return spin::fail(SPIN_ERR_MEMORY, "device allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
        SPIN_CUDA(cudaMemsetAsync(*a, 0, bytes, s->stream));      // ghost cells of open edges must read as zero forever
    }
    s->cur = 0;
    if (keep) {
        int *bad = (int *)(s->d_aos + (size_t)3 * s->N);
        for (int k = 0; k < s->n_img; ++k)
            pack_kernel<<<nblk, nt, 0, s->stream>>>(P, stage + (size_t)k * 3 * s->N, s->d_n[0] + (size_t)k * s->nb * P.sub, (int)s->N, 0, bad);
        s->n_launch += s->n_img;
    }
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    if (stage != s->d_aos) cudaFree(stage);
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

// per-image factor on the thermal amplitude, sqrt(T_image / T), from the absolute image temperatures kept on the host; called whenever
// either side of the ratio changes (llg_set_image_temperatures, llg_configure through ensure_plan)
int upload_image_sigma(spin_system *s) {
    if (s->img_T.empty()) return SPIN_OK;
    if (!(s->T > 0.0)) return spin::fail(SPIN_ERR_STATE, "per-image temperatures are set but the reference temperature of llg_configure is 0: set T > 0 or clear them");
    if ((int)s->img_T.size() != s->n_img) return spin::fail(SPIN_ERR_STATE, "per-image temperatures were set for %d images, the system has %d", (int)s->img_T.size(), s->n_img);
    std::vector<double> sc((size_t)s->n_img);
    for (int k = 0; k < s->n_img; ++k) sc[(size_t)k] = sqrt(s->img_T[(size_t)k] / s->T);
    if (!s->d_img_sigma) SPIN_CUDA(cudaMalloc(&s->d_img_sigma, (size_t)s->n_img * sizeof(double)));
    SPIN_CUDA(cudaMemcpyAsync(s->d_img_sigma, sc.data(), (size_t)s->n_img * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    drop_graphs(s);                           // captured launches hold the old pointer
    return SPIN_OK;
}

// mu_i / mu_b(i) in boundary order from the per-site moments kept on the host
int upload_mu_ratio(spin_system *s) {
    if (s->mu_site.empty()) return SPIN_OK;
    std::vector<double> r((size_t)s->N);
    for (int64_t i = 0; i < s->N; ++i) r[(size_t)i] = s->mu_site[(size_t)i] / s->mu[(size_t)(i % s->nb)];
    if (!s->d_mu_ratio) {
        cudaError_t e = cudaMalloc(&s->d_mu_ratio, (size_t)s->N * sizeof(double));
        if (e != cudaSuccess) { s->d_mu_ratio = nullptr; return spin::fail(SPIN_ERR_MEMORY, "device allocation of %lld bytes failed", (long long)(s->N * 8)); }
    }
    SPIN_CUDA(cudaMemcpyAsync(s->d_mu_ratio, r.data(), (size_t)s->N * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    return SPIN_OK;
}

int ensure_plan(spin_system *s) {
    NEED_DEVICE(s);
    if (!s->plan_dirty) return SPIN_OK;
    s->vp_active = false;
    int rc = upload_mu_ratio(s);               // per-site moments relative to the (possibly changed) basis moments
    if (rc) return rc;
    DevicePlan P;
    rc = build_plan(s, P);
    if (rc) return rc;
    drop_graphs(s);
    if (!s->d_n[0] || !same_layout(P, s->plan)) {
        rc = allocate_arrays(s, P, s->d_n[0] != nullptr);
        if (rc) return rc;
    }
    s->plan = P;
    rc = upload_image_sigma(s);               // T may have changed: the ratios sqrt(T_image / T) follow
    if (rc) return rc;
    if (s->ddi_on) {
        rc = ddi_prepare(s);
        if (rc) return rc;
    } else {
        ddi_release(s);
    }
    // run-time specialised sweeps; on failure the table-driven kernels stay in use and the reason is kept
    s->jit_note.clear();
    if (s->opt_jit) {
        rc = jit_prepare(s);
        if (rc) { s->jit_note = spin_last_error(); jit_release(s); }
    } else {
        jit_release(s);
        s->jit_note = "disabled by option use_jit=0";
    }
    s->plan_dirty = false;
    return SPIN_OK;
}

// one Depondt step enqueued on the stream; step_add is added to the device step counter by the kernels
template <int BX, int BY, int BZ>
int enqueue_step_t(spin_system *s, const Launch &L, unsigned step_add) {
    double *n = s->d_n[s->cur], *nout = s->d_n[s->cur ^ 1];
    if (s->solver == SPIN_SOLVER_RK4) {
        // four field sweeps: stage configurations in d_np / d_fddi[1], weighted sum of the k in d_A, thermal field of the step in
        // d_fddi[0] (lattices without dipolar coupling; with it d_fddi[0] holds the dipolar field of the stage configuration)
        const double *y[4] = {n, s->d_np, s->d_fddi[1], s->d_np};
        double *yn[4] = {s->d_np, s->d_fddi[1], s->d_np, nout};
        for (int st = 0; st < 4; ++st) {
            if (s->ddi_on) { int rc = ddi_field(s, y[st], s->d_fddi[0]); if (rc) return rc; }
            int rc = jit_launch_rk4_stage(s, n, y[st], yn[st], s->d_A, s->d_fddi[0], s->d_fddi[0], st, step_add);
            if (rc) return rc;
            s->n_launch++;
        }
        s->cur ^= 1;
        return SPIN_OK;
    }
    const bool prof = s->profile_on != 0;
    if (jit_march_ready(s)) {          // the whole step in one pass (n^p stays in shared memory)
        if (prof) cudaEventRecord(s->ev0, s->stream);
        int rc = jit_launch_march(s, s->cur, nout, step_add);
        if (rc) return rc;
        s->n_launch++;
        if (prof) { cudaEventRecord(s->ev1, s->stream); cudaEventSynchronize(s->ev1); float ms; cudaEventElapsedTime(&ms, s->ev0, s->ev1); s->prof_ms[1] += ms; s->prof_n[1]++; }
        s->cur ^= 1;
        return SPIN_OK;
    }
    const size_t istr = (size_t)s->nb * s->plan.sub;       // image stride
    if (s->ddi_on) {
        if (prof) cudaEventRecord(s->ev0, s->stream);
        int rc = SPIN_OK;
        for (int k = 0; k < s->n_img && rc == SPIN_OK; ++k) rc = ddi_field(s, n + k * istr, s->d_fddi[0] + k * istr);
        if (rc) return rc;
        if (prof) { cudaEventRecord(s->ev1, s->stream); cudaEventSynchronize(s->ev1); float ms; cudaEventElapsedTime(&ms, s->ev0, s->ev1); s->prof_ms[2] += ms; s->prof_n[2]++; }
    }
    const bool jit = jit_ready(s);
    if (prof) cudaEventRecord(s->ev0, s->stream);
    if (jit) { int rc = jit_launch_predictor(s, L.grid, L.block, n, s->d_fddi[0], s->d_np, s->d_A, step_add); if (rc) return rc; }
    else if (s->opt_store_A)
        predictor_kernel<BX, BY, BZ, true><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], s->d_np, s->d_A, s->d_step, step_add);
    else
        predictor_kernel<BX, BY, BZ, false><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], s->d_np, nullptr, s->d_step, step_add);
    s->n_launch++;
    if (prof) { cudaEventRecord(s->ev1, s->stream); cudaEventSynchronize(s->ev1); float ms; cudaEventElapsedTime(&ms, s->ev0, s->ev1); s->prof_ms[0] += ms; s->prof_n[0]++; }
    if (s->ddi_on) {
        if (prof) cudaEventRecord(s->ev0, s->stream);
        int rc = SPIN_OK;
        for (int k = 0; k < s->n_img && rc == SPIN_OK; ++k) rc = ddi_field(s, s->d_np + k * istr, s->d_fddi[1] + k * istr);
        if (rc) return rc;
        if (prof) { cudaEventRecord(s->ev1, s->stream); cudaEventSynchronize(s->ev1); float ms; cudaEventElapsedTime(&ms, s->ev0, s->ev1); s->prof_ms[2] += ms; s->prof_n[2]++; }
    }
    if (prof) cudaEventRecord(s->ev0, s->stream);
    if (jit) { int rc = jit_launch_corrector(s, L.grid, L.block, n, s->d_np, s->d_fddi[0], s->d_fddi[1], s->d_A, nout, step_add); if (rc) return rc; }
    else if (s->opt_store_A)
        corrector_kernel<BX, BY, BZ, true><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_np, s->d_fddi[0], s->d_fddi[1], s->d_A, nout, s->d_step, step_add);
    else
        corrector_kernel<BX, BY, BZ, false><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_np, s->d_fddi[0], s->d_fddi[1], nullptr, nout, s->d_step, step_add);
    s->n_launch++;
    if (prof) { cudaEventRecord(s->ev1, s->stream); cudaEventSynchronize(s->ev1); float ms; cudaEventElapsedTime(&ms, s->ev0, s->ev1); s->prof_ms[1] += ms; s->prof_n[1]++; }
    s->cur ^= 1;
    return SPIN_OK;
}
int enqueue_step(spin_system *s, unsigned step_add) {
    const Launch L = brick_launch(s);
    return L.flat ? enqueue_step_t<32, 8, 1>(s, L, step_add) : enqueue_step_t<32, 4, 2>(s, L, step_add);
}

// deterministic force of the current configuration into d_np (scratch), terms by mask
int enqueue_force(spin_system *s, int mask, double *d_out) {
    const Launch L = brick_launch(s);
    double *n = s->d_n[s->cur] + img_off(s);
    if (s->ddi_on && (mask & T_DDI)) { int rc = ddi_field(s, n, s->d_fddi[0]); if (rc) return rc; }
    if (L.flat) force_kernel<32, 8, 1><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], mask, d_out);
    else force_kernel<32, 4, 2><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], mask, d_out);
    s->n_launch++;
    return SPIN_OK;
}

// the N_RED reductions of the selected image into d_out (device), no synchronisation
int enqueue_reduce(spin_system *s, double *d_out) {
    const Launch L = brick_launch(s);
    double *n = s->d_n[s->cur] + img_off(s);
    if (s->ddi_on) { int rc = ddi_field(s, n, s->d_fddi[0]); if (rc) return rc; }
    const int nblocks = (int)(L.grid.x * L.grid.y);
    if (L.flat) reduce_kernel<32, 8, 1><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], s->d_partials);
    else reduce_kernel<32, 4, 2><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], s->d_partials);
    reduce_final_kernel<<<1, 32 * N_RED, 0, s->stream>>>(s->d_partials, nblocks, d_out);
    s->n_launch += 2;
    return SPIN_OK;
}

int reduce_all(spin_system *s, double out[N_RED]) {
    int rc = enqueue_reduce(s, s->d_result);
    if (rc) return rc;
    SPIN_CUDA(cudaMemcpyAsync(out, s->d_result, N_RED * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------- lifecycle
extern "C" int spin_geometry_create(const double bravais[9], int n_basis, const double *basis_frac, const int n_cells[3],
                                    const int periodic[3], double lattice_constant_A, spin_system **out) {
    REQUIRE(bravais && basis_frac && n_cells && periodic && out, "null argument");
    REQUIRE(n_basis >= 1 && n_basis <= SPIN_MAX_BASIS, "n_basis must be in [1, %d]", SPIN_MAX_BASIS);
    REQUIRE(lattice_constant_A > 0.0, "lattice constant must be positive");
    int64_t ncell = 1;
    for (int d = 0; d < 3; ++d) { REQUIRE(n_cells[d] >= 1, "n_cells must be >= 1"); ncell *= n_cells[d]; }
    REQUIRE(ncell * n_basis < (int64_t)2147483647 / 3, "lattice too large for 32-bit indexing");
    const double *a = bravais, *b = bravais + 3, *c = bravais + 6;
    const double vol = a[0] * (b[1] * c[2] - b[2] * c[1]) - a[1] * (b[0] * c[2] - b[2] * c[0]) + a[2] * (b[0] * c[1] - b[1] * c[0]);
    REQUIRE(fabs(vol) > 1e-12, "bravais vectors are linearly dependent");
    int ndev = 0;
    bool has_device = cudaGetDeviceCount(&ndev) == cudaSuccess && ndev >= 1;
    // planner-only mode for the CPU test-suite (gather tables, generated kernel source); nothing can be computed in it
    const char *plan_only = getenv("SPINLLG_PLANNER_ONLY");
    if (!has_device && !(plan_only && plan_only[0] == '1'))
        return spin::fail(SPIN_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    if (!has_device) cudaGetLastError();
    spin_system *s = new spin_system();
    s->has_device = has_device;
    s->jit = nullptr; s->opt_jit = 1; s->opt_march = 1; s->opt_ddi_slab = 1; s->opt_ddi_mirror = 1; s->opt_pdl = -1; s->opt_cache_noise = 1; s->opt_coop = 1; s->d_bar = nullptr; s->d_flags = nullptr;
    s->n_img = 1; s->img_sel = 0; s->d_img_sigma = nullptr;
    memcpy(s->brav, bravais, sizeof(s->brav));
    s->nb = n_basis;
    s->basis.assign(basis_frac, basis_frac + 3 * n_basis);
    for (int d = 0; d < 3; ++d) { s->nc[d] = n_cells[d]; s->per[d] = periodic[d] ? 1 : 0; }
    s->alat = lattice_constant_A;
    s->ncell = ncell; s->N = ncell * n_basis;
    s->mu.assign(n_basis, 1.0);
    s->Bmag = 0.0; s->Bdir[0] = 0; s->Bdir[1] = 0; s->Bdir[2] = 1;
    s->ani_b.clear(); s->K.clear(); s->Kax.clear();
    s->ddi_on = 0; s->ddi_img[0] = s->ddi_img[1] = s->ddi_img[2] = 0;
    s->dt_ps = 1e-3; s->alpha = 0.1; s->T = 0; s->u = 0; s->jdir[0] = 1; s->jdir[1] = 0; s->jdir[2] = 0; s->beta = 0;
    s->seed = 0; s->step = 0; s->solver = SPIN_SOLVER_DEPONDT; s->damping_only = 0;
    s->stream = nullptr; s->own_stream = nullptr; s->cur = 0;
    s->d_n[0] = s->d_n[1] = s->d_np = s->d_A = s->d_fddi[0] = s->d_fddi[1] = s->d_aos = s->d_partials = s->d_result = nullptr;
    s->d_vp = nullptr; s->vp_active = false; s->vp_cur = 0;
    s->slab_on = 0; s->slab_off = 0; s->slab_gnc = 0; s->slab_gper = 0;
    s->d_step = nullptr; s->d_pin = nullptr; s->d_mu_ratio = nullptr; s->ddi = nullptr; s->plan_dirty = true;
    s->opt_graph = 1; s->opt_store_A = 0; s->graph_exec[0] = s->graph_exec[1] = nullptr; s->graph_steps = 0;
    s->n_launch = s->n_fft = 0; s->profile_on = 0;
    for (int k = 0; k < 3; ++k) { s->prof_ms[k] = 0; s->prof_n[k] = 0; }
    s->ev0 = s->ev1 = s->ev2 = s->ev3 = nullptr;
    const Launch L = brick_launch(s);
    memset(&s->plan, 0, sizeof(s->plan));
    if (!has_device) { *out = s; return SPIN_OK; }
    cudaError_t e = cudaStreamCreateWithFlags(&s->own_stream, cudaStreamNonBlocking);
    s->stream = s->own_stream;
    if (e == cudaSuccess) e = cudaMalloc(&s->d_aos, (size_t)3 * s->N * sizeof(double) + sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_partials, (size_t)L.grid.x * L.grid.y * N_RED * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_result, 16 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_vp, 4 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_bar, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_step, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(s->d_step, 0, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaEventCreate(&s->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&s->ev1);
    if (e == cudaSuccess) e = cudaEventCreate(&s->ev2);
    if (e == cudaSuccess) e = cudaEventCreate(&s->ev3);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        const int code = (e == cudaErrorMemoryAllocation) ? SPIN_ERR_MEMORY : SPIN_ERR_CUDA;
        spin::fail(code, "device setup failed: %s", cudaGetErrorString(e));
        spin_system_destroy(s);
        return code;
    }
    // address of the fixed scratch array of topological_charge_noalloc on this device (resolved once per device; a failure is reported
    // by that entry point, the only one that needs it)
    if (topo_noalloc_setup() != SPIN_OK) cudaGetLastError();
    // initial state: all spins +z
    std::vector<double> z((size_t)3 * s->N, 0.0);
    for (int64_t i = 0; i < s->N; ++i) z[3 * i + 2] = 1.0;
    *out = s;
    DevicePlan P0;                    // initial layout (no interactions yet: no ghost cells); the plan stays dirty
    int rc = build_plan(s, P0);
    if (rc == SPIN_OK) rc = allocate_arrays(s, P0, false);
    if (rc == SPIN_OK) { s->plan = P0; rc = spins_set(s, z.data()); }
    if (rc) { spin_system_destroy(s); *out = nullptr; return rc; }
    return SPIN_OK;
}

extern "C" void spin_system_destroy(spin_system *s) {
    if (!s) return;
    drop_graphs(s);
    if (s->own_stream) cudaStreamDestroy(s->own_stream);
    ddi_release(s);
    jit_release(s);
    cudaFree(s->d_n[0]); cudaFree(s->d_n[1]); cudaFree(s->d_np); cudaFree(s->d_A); cudaFree(s->d_fddi[0]); cudaFree(s->d_fddi[1]);
    cudaFree(s->d_pin); cudaFree(s->d_vp); cudaFree(s->d_bar); cudaFree(s->d_img_sigma); cudaFree(s->d_flags);
    cudaFree(s->d_aos); cudaFree(s->d_partials); cudaFree(s->d_result); cudaFree(s->d_step); cudaFree(s->d_mu_ratio);
    if (s->ev0) cudaEventDestroy(s->ev0);
    if (s->ev1) cudaEventDestroy(s->ev1);
    if (s->ev2) cudaEventDestroy(s->ev2);
    if (s->ev3) cudaEventDestroy(s->ev3);
    delete s;
}

extern "C" int64_t spin_system_nspins(const spin_system *s) { return s ? s->N : 0; }

extern "C" int spin_set_stream(spin_system *s, void *stream) {
    REQUIRE(s, "null system");
    NEED_DEVICE(s);
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    s->stream = stream ? (cudaStream_t)stream : s->own_stream;
    drop_graphs(s);
    if (s->ddi) s->plan_dirty = true;     // cuFFT plans are bound to a stream
    return SPIN_OK;
}

// ---------------------------------------------------------------------------------------------- Hamiltonian setters
extern "C" int hamiltonian_set_mu_s(spin_system *s, const double *mu) {
    REQUIRE(s && mu, "null argument");
    for (int b = 0; b < s->nb; ++b) REQUIRE(mu[b] > 0.0 && isfinite(mu[b]), "mu_s must be positive");
    s->mu.assign(mu, mu + s->nb);
    s->plan_dirty = true;
    return SPIN_OK;
}
// PAPER.md:79 "defects, such as vacancies and atoms of different types": a moment per site (mu_B, boundary order) that replaces the basis
// atom's wherever mu_i enters: Zeeman force, dipolar sums, the 1/mu_i of Eq. 10, the thermal amplitude of Eq. 11, the conversion to Tesla
extern "C" int hamiltonian_set_site_mu_s(spin_system *s, const double *mu_site) {
    REQUIRE(s, "null system");
    if (!mu_site) {
        s->mu_site.clear();
        if (s->d_mu_ratio) { if (s->has_device) cudaStreamSynchronize(s->stream); cudaFree(s->d_mu_ratio); s->d_mu_ratio = nullptr; }
    } else {
        for (int64_t i = 0; i < s->N; ++i) REQUIRE(mu_site[i] > 0.0 && isfinite(mu_site[i]), "site %lld: moment must be positive and finite", (long long)i);
        s->mu_site.assign(mu_site, mu_site + s->N);
    }
    s->plan_dirty = true;
    drop_graphs(s);
    return SPIN_OK;
}
extern "C" int hamiltonian_set_field(spin_system *s, double B, const double dir[3]) {
    REQUIRE(s && dir, "null argument");
    const double n = sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
    REQUIRE(isfinite(B) && (n > 0.0 || B == 0.0), "field direction must be non-zero");
    s->Bmag = B;
    for (int k = 0; k < 3; ++k) s->Bdir[k] = n > 0.0 ? dir[k] / n : (k == 2 ? 1.0 : 0.0);
    s->plan_dirty = true;
    return SPIN_OK;
}
extern "C" int hamiltonian_set_anisotropy(spin_system *s, int n, const int *bidx, const double *K, const double *axis) {
    REQUIRE(s && n >= 0 && (n == 0 || (bidx && K && axis)), "bad argument");
    REQUIRE(n <= SPIN_MAX_ANI_ENTRIES, "at most %d anisotropy axes in total", SPIN_MAX_ANI_ENTRIES);
    std::vector<int> ab;
    std::vector<double> Kn, ax;
    for (int e = 0; e < n; ++e) {
        REQUIRE(bidx[e] >= 0 && bidx[e] < s->nb, "anisotropy: basis index %d out of range", bidx[e]);
        const double *a = axis + 3 * e;
        const double nn = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
        REQUIRE(nn > 0.0 && isfinite(K[e]), "anisotropy: zero axis or non-finite K");
        ab.push_back(bidx[e]);
        Kn.push_back(K[e]);
        for (int k = 0; k < 3; ++k) ax.push_back(a[k] / nn);
    }
    s->ani_b = ab; s->K = Kn; s->Kax = ax;
    s->plan_dirty = true;
    return SPIN_OK;
}
extern "C" int hamiltonian_set_pairs(spin_system *s, int np, const int *bi, const int *bj, const int *t, const double *J, const double *D) {
    REQUIRE(s && np >= 0 && (np == 0 || (bi && bj && t && J)), "bad argument");
    std::vector<HostPair> v;
    std::map<std::vector<int>, int> seen;
    for (int p = 0; p < np; ++p) {
        REQUIRE(bi[p] >= 0 && bi[p] < s->nb && bj[p] >= 0 && bj[p] < s->nb, "pair %d: basis index out of range", p);
        REQUIRE(!(bi[p] == bj[p] && t[3 * p] == 0 && t[3 * p + 1] == 0 && t[3 * p + 2] == 0), "pair %d couples a site with itself", p);
        // the same bond listed in both directions would be double counting (":69 unique pairs")
        std::vector<int> fwd = {bi[p], bj[p], t[3 * p], t[3 * p + 1], t[3 * p + 2]}, bwd = {bj[p], bi[p], -t[3 * p], -t[3 * p + 1], -t[3 * p + 2]};
        REQUIRE(!seen.count(bwd) || fwd == bwd, "pair %d repeats pair %d in the opposite direction", p, seen.count(bwd) ? seen[bwd] : -1);
        seen[fwd] = p;
        HostPair h;
        h.bi = bi[p]; h.bj = bj[p];
        for (int k = 0; k < 3; ++k) { h.t[k] = t[3 * p + k]; h.D[k] = D ? D[3 * p + k] : 0.0; }
        h.J = J[p];
        REQUIRE(isfinite(h.J) && isfinite(h.D[0]) && isfinite(h.D[1]) && isfinite(h.D[2]), "pair %d: non-finite coupling", p);
        v.push_back(h);
    }
    s->pairs_explicit.swap(v);
    s->plan_dirty = true;
    return SPIN_OK;
}
extern "C" int hamiltonian_set_exchange_shells(spin_system *s, int n_shells, const double *J) {
    REQUIRE(s && n_shells >= 0 && (n_shells == 0 || J), "bad argument");
    std::vector<HostPair> v;
    if (n_shells > 0) {
        auto shells = find_shells(s, n_shells);
        REQUIRE((int)shells.size() == n_shells, "only %d neighbour shells exist on this lattice", (int)shells.size());
        for (int k = 0; k < n_shells; ++k)
            for (const Bond &b : shells[k]) {
                HostPair h;
                h.bi = b.bi; h.bj = b.bj; h.J = J[k];
                for (int d = 0; d < 3; ++d) { h.t[d] = b.t[d]; h.D[d] = 0.0; }
                v.push_back(h);
            }
    }
    s->pairs_exch_shells.swap(v);
    s->plan_dirty = true;
    return SPIN_OK;
}
extern "C" int hamiltonian_set_dmi_shells(spin_system *s, int n_shells, const double *Dm, int chirality) {
    REQUIRE(s && n_shells >= 0 && (n_shells == 0 || Dm), "bad argument");
    REQUIRE(chirality == 1 || chirality == -1 || chirality == 2 || chirality == -2, "chirality must be +-1 (bulk) or +-2 (interfacial)");
    std::vector<HostPair> v;
    if (n_shells > 0) {
        auto shells = find_shells(s, n_shells);
        REQUIRE((int)shells.size() == n_shells, "only %d neighbour shells exist on this lattice", (int)shells.size());
        for (int k = 0; k < n_shells; ++k)
            for (const Bond &b : shells[k]) {
                HostPair h;
                h.bi = b.bi; h.bj = b.bj; h.J = 0.0;
                const double rh[3] = {b.r[0] / b.len, b.r[1] / b.len, b.r[2] / b.len};
                const double sg = chirality > 0 ? 1.0 : -1.0;
                if (abs(chirality) == 1) { h.D[0] = sg * Dm[k] * rh[0]; h.D[1] = sg * Dm[k] * rh[1]; h.D[2] = sg * Dm[k] * rh[2]; }
                else { h.D[0] = sg * Dm[k] * (-rh[1]); h.D[1] = sg * Dm[k] * rh[0]; h.D[2] = 0.0; }      // z x r
                for (int d = 0; d < 3; ++d) h.t[d] = b.t[d];
                v.push_back(h);
            }
    }
    s->pairs_dmi_shells.swap(v);
    s->plan_dirty = true;
    return SPIN_OK;
}
extern "C" int hamiltonian_set_quadruplets(spin_system *s, int n, const int *b4, const int *t9, const double *K) {
    REQUIRE(s && n >= 0 && (n == 0 || (b4 && t9 && K)), "bad argument");
    std::vector<HostQuad> v;
    for (int q = 0; q < n; ++q) {
        HostQuad h;
        for (int k = 0; k < 4; ++k) { h.b[k] = b4[4 * q + k]; REQUIRE(h.b[k] >= 0 && h.b[k] < s->nb, "quadruplet %d: basis index out of range", q); }
        for (int k = 0; k < 9; ++k) h.t[k] = t9[9 * q + k];
        h.K = K[q];
        REQUIRE(isfinite(h.K), "quadruplet %d: non-finite K", q);
        v.push_back(h);
    }
    s->quads.swap(v);
    s->plan_dirty = true;
    return SPIN_OK;
}
extern "C" int hamiltonian_set_ddi(spin_system *s, int enabled, const int img[3]) {
    REQUIRE(s && (!enabled || img), "bad argument");
    if (enabled) for (int d = 0; d < 3; ++d) REQUIRE(img[d] >= 0 && img[d] <= 1000, "n_periodic_images out of range");
    s->ddi_on = enabled ? 1 : 0;
    for (int d = 0; d < 3; ++d) s->ddi_img[d] = enabled ? img[d] : 0;
    s->plan_dirty = true;
    return SPIN_OK;
}

// ---------------------------------------------------------------------------------------------- state
static int pack_from_device_aos(spin_system *s, const double *d_aos) {
    NEED_DEVICE(s);
    s->vp_active = false;
    int *bad = (int *)(s->d_aos + (size_t)3 * s->N);
    SPIN_CUDA(cudaMemsetAsync(bad, 0, sizeof(int), s->stream));
    const int nt = 256;
    pack_kernel<<<(unsigned)((s->N + nt - 1) / nt), nt, 0, s->stream>>>(s->plan, d_aos, s->d_n[s->cur] + img_off(s), (int)s->N, 1, bad);
    s->n_launch++;
    int h_bad = 0;
    SPIN_CUDA(cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    SPIN_CUDA(cudaGetLastError());
    if (h_bad) return spin::fail(SPIN_ERR_ARG, "spins_set: zero or non-finite spin vector");
    return SPIN_OK;
}
// ---- batched images
extern "C" int spin_set_images(spin_system *s, int n_images) {
    REQUIRE(s && n_images >= 1 && n_images <= 65535, "n_images must be in [1, 65535]");
    NEED_DEVICE(s);
    if (n_images == s->n_img) return SPIN_OK;
    int rc = ensure_plan(s);                  // settle the layout first
    if (rc) return rc;
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    const size_t istr = (size_t)s->nb * s->plan.sub, ibytes = istr * sizeof(double);
    const int n_old = s->n_img, n_keep = std::min(n_old, n_images);
    double *old = nullptr;
    SPIN_CUDA(cudaMalloc(&old, (size_t)n_old * ibytes));
    {   // every copy goes through the system's stream (a device-to-device cudaMemcpy on the legacy stream is not ordered with it)
        cudaError_t e = cudaMemcpyAsync(old, s->d_n[s->cur], (size_t)n_old * ibytes, cudaMemcpyDeviceToDevice, s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) { cudaFree(old); return spin::fail(SPIN_ERR_CUDA, "spin_set_images: %s", cudaGetErrorString(e)); }
    }
    s->n_img = n_images;
    s->img_sel = 0;
    rc = allocate_arrays(s, s->plan, false);
    if (rc == SPIN_OK) {
        cudaError_t e = cudaMemcpyAsync(s->d_n[0], old, (size_t)n_keep * ibytes, cudaMemcpyDeviceToDevice, s->stream);
        for (int k = n_keep; k < n_images && e == cudaSuccess; ++k)      // new images start as copies of image 0
            e = cudaMemcpyAsync(s->d_n[0] + (size_t)k * istr, old, ibytes, cudaMemcpyDeviceToDevice, s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) rc = spin::fail(SPIN_ERR_CUDA, "spin_set_images: %s", cudaGetErrorString(e));
    }
    cudaFree(old);
    if (s->d_img_sigma) { cudaFree(s->d_img_sigma); s->d_img_sigma = nullptr; }
    s->img_T.clear();                         // per-image temperatures belong to the old image count
    s->plan_dirty = true;                     // kernels variants and dipolar buffers depend on the image count
    drop_graphs(s);
    return rc;
}
extern "C" int spin_select_image(spin_system *s, int image) {
    REQUIRE(s && image >= 0 && image < s->n_img, "image index out of range");
    s->img_sel = image;
    return SPIN_OK;
}
extern "C" int llg_set_image_temperatures(spin_system *s, const double *T_kelvin) {
    REQUIRE(s, "null system");
    NEED_DEVICE(s);
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    if (!T_kelvin) { s->img_T.clear(); if (s->d_img_sigma) { cudaFree(s->d_img_sigma); s->d_img_sigma = nullptr; } drop_graphs(s); return SPIN_OK; }
    REQUIRE(s->T > 0.0, "llg_configure must set a positive reference temperature first");
    for (int k = 0; k < s->n_img; ++k) REQUIRE(T_kelvin[k] >= 0.0 && isfinite(T_kelvin[k]), "image %d: temperature must be >= 0", k);
    s->img_T.assign(T_kelvin, T_kelvin + s->n_img);      // absolute temperatures: the scale array follows later changes of T
    return upload_image_sigma(s);
}

// pinned spins: flags in boundary order; null clears.  A pinned site may hold the zero vector (a vacancy).
extern "C" int spins_set_pinned(spin_system *s, const unsigned char *mask) {
    REQUIRE(s, "null system");
    NEED_DEVICE(s);
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    if (!mask) {
        if (s->d_pin) { cudaFree(s->d_pin); s->d_pin = nullptr; }
    } else {
        if (!s->d_pin) {
            cudaError_t e = cudaMalloc(&s->d_pin, (size_t)s->N);
            if (e != cudaSuccess) { s->d_pin = nullptr; return spin::fail(SPIN_ERR_MEMORY, "device allocation of %lld bytes failed", (long long)s->N); }
        }
        SPIN_CUDA(cudaMemcpyAsync(s->d_pin, mask, (size_t)s->N, cudaMemcpyHostToDevice, s->stream));
        SPIN_CUDA(cudaStreamSynchronize(s->stream));
    }
    s->plan.pin = s->d_pin;       // pack_kernel reads it before the next plan build
    s->plan_dirty = true;
    drop_graphs(s);
    return SPIN_OK;
}
extern "C" int spins_set(spin_system *s, const double *n) {
    REQUIRE(s && n, "null argument");
    NEED_DEVICE(s);
    SPIN_CUDA(cudaMemcpyAsync(s->d_aos, n, (size_t)3 * s->N * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    return pack_from_device_aos(s, s->d_aos);
}
extern "C" int spins_set_device(spin_system *s, const double *n) {
    REQUIRE(s && n, "null argument");
    return pack_from_device_aos(s, n);
}
extern "C" int spins_get_device(spin_system *s, double *n) {
    REQUIRE(s && n, "null argument");
    NEED_DEVICE(s);
    const int nt = 256;
    unpack_kernel<<<(unsigned)((s->N + nt - 1) / nt), nt, 0, s->stream>>>(s->plan, s->d_n[s->cur] + img_off(s), n, (int)s->N, 0);
    s->n_launch++;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
extern "C" int spins_get(spin_system *s, double *n) {
    REQUIRE(s && n, "null argument");
    int rc = spins_get_device(s, s->d_aos);
    if (rc) return rc;
    SPIN_CUDA(cudaMemcpyAsync(n, s->d_aos, (size_t)3 * s->N * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    return SPIN_OK;
}

// ---------------------------------------------------------------------------------------------- dynamics
extern "C" int llg_configure(spin_system *s, double dt_fs, double alpha, double T, uint64_t seed, double u, const double jdir[3], double beta) {
    REQUIRE(s, "null system");
    REQUIRE(dt_fs > 0.0 && isfinite(dt_fs), "dt must be positive");
    REQUIRE(alpha >= 0.0 && isfinite(alpha), "alpha must be >= 0");
    REQUIRE(T >= 0.0 && isfinite(T), "T must be >= 0");
    REQUIRE(isfinite(u) && isfinite(beta), "non-finite current parameters");
    double j[3] = {1, 0, 0};
    if (jdir) { j[0] = jdir[0]; j[1] = jdir[1]; j[2] = jdir[2]; }
    const double nn = sqrt(j[0] * j[0] + j[1] * j[1] + j[2] * j[2]);
    REQUIRE(nn > 0.0 || u == 0.0, "current direction must be non-zero");
    s->dt_ps = dt_fs * 1e-3; s->alpha = alpha; s->T = T; s->seed = seed; s->u = u; s->beta = beta;
    for (int k = 0; k < 3; ++k) s->jdir[k] = nn > 0.0 ? j[k] / nn : (k == 0 ? 1.0 : 0.0);
    s->plan_dirty = true;
    return llg_set_step(s, 0);
}
extern "C" int llg_set_solver(spin_system *s, int solver) {
    REQUIRE(s, "null system");
    REQUIRE(solver == SPIN_SOLVER_DEPONDT || solver == SPIN_SOLVER_HEUN || solver == SPIN_SOLVER_SIB || solver == SPIN_SOLVER_RK4, "unknown solver %d", solver);
    if (s->solver != solver) { s->solver = solver; s->plan_dirty = true; drop_graphs(s); }
    return SPIN_OK;
}
extern "C" int llg_set_damping_only(spin_system *s, int enabled) {
    REQUIRE(s, "null system");
    if (s->damping_only != (enabled ? 1 : 0)) { s->damping_only = enabled ? 1 : 0; s->plan_dirty = true; drop_graphs(s); }
    return SPIN_OK;
}
extern "C" int llg_get_step(const spin_system *s, uint64_t *step) {
    REQUIRE(s && step, "null argument");
    *step = s->step;
    return SPIN_OK;
}
extern "C" int llg_set_step(spin_system *s, uint64_t step) {
    REQUIRE(s, "null system");
    s->step = step;
    if (!s->has_device) return SPIN_OK;
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    const unsigned long long v = step;
    SPIN_CUDA(cudaMemcpyAsync(s->d_step, &v, sizeof(v), cudaMemcpyHostToDevice, s->stream));      // ordered on the system's stream, like the sweeps
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    return SPIN_OK;
}

extern "C" int llg_iterate(spin_system *s, int64_t n_steps) {
    REQUIRE(s && n_steps >= 0, "bad argument");
    int rc = ensure_plan(s);
    if (rc) return rc;
    if (s->slab_on) return spin::fail(SPIN_ERR_STATE, "a slab advances through llg_slab_sweep / spin_halo_* / llg_slab_advance (its ghost layers need the halo exchange)");
    s->vp_active = false;
    if (s->n_img > 1 && (!jit_ready(s) || s->solver == SPIN_SOLVER_RK4))
        return spin::fail(SPIN_ERR_STATE, "batched images need the run-time specialised kernels and a two-stage solver (%s)", s->jit_note.c_str());
    if (s->solver != SPIN_SOLVER_DEPONDT && !jit_ready(s))
        return spin::fail(SPIN_ERR_STATE, "the Heun, SIB and RK4 solvers need the run-time specialised kernels (%s)", s->jit_note.c_str());
    int64_t done = 0;
    // The smallest lattices (a handful of blocks): all steps in one cooperative launch, in chunks that keep the barrier counter far
    // from wrapping.  Measured on B200: 4.33 vs 4.61 us per step at 1,024 spins, but 5.29 vs 5.12 at 16,384 and 13.8 vs 10.4 at 65,536
    // (a grid barrier costs about as much as a launch inside a CUDA graph, and it empties L1), so the limit is low; option
    // use_coop = 2 forces it for any lattice without dipolar coupling.
    const int64_t COOP_CHUNK = 8192;
    if (s->opt_coop && !s->profile_on && !s->ddi_on && (s->N <= SPIN_COOP_MAX_SPINS || s->opt_coop >= 2) && jit_coop_ready(s) && !jit_march_ready(s) &&
        n_steps > 0) {
        while (done < n_steps) {
            const unsigned chunk = (unsigned)std::min<int64_t>(COOP_CHUNK, n_steps - done);
            rc = jit_launch_steps_coop(s, chunk);
            if (rc) return rc;
            advance_step_kernel<<<1, 1, 0, s->stream>>>(s->d_step, (unsigned long long)chunk);
            s->n_launch += 2;
            if (chunk & 1u) s->cur ^= 1;
            done += chunk;
        }
        s->step += (uint64_t)n_steps;
        SPIN_CUDA(cudaGetLastError());
        return SPIN_OK;
    }
    // Larger lattices: replay a captured graph of G steps (an even number, so the ping-pong buffers return to the
    // same roles); the kernels read the step counter from device memory, the graph's last node advances it by G.
    // (dipolar coupling: only the path that is kernels throughout -- cuFFT's transforms stay outside a capture)
    const bool graph_ok = s->opt_graph && !s->profile_on && (!s->ddi_on || ddi_graph_ok(s));
    const int G = 16;
    if (graph_ok && n_steps >= G) {
        cudaGraphExec_t &gexec = s->graph_exec[s->cur];
        if (!gexec) {
            cudaGraph_t graph = nullptr;
            SPIN_CUDA(cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
            const int64_t launches_before = s->n_launch;
            for (int k = 0; k < G && rc == SPIN_OK; ++k) rc = enqueue_step(s, (unsigned)k);
            advance_step_kernel<<<1, 1, 0, s->stream>>>(s->d_step, (unsigned long long)G);
            s->graph_launches = s->n_launch - launches_before + 1;      // what one replay launches
            s->n_launch = launches_before;
            cudaError_t e = cudaStreamEndCapture(s->stream, &graph);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return spin::fail(SPIN_ERR_CUDA, "graph capture failed: %s", cudaGetErrorString(e));
            e = cudaGraphInstantiate(&gexec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { gexec = nullptr; return spin::fail(SPIN_ERR_CUDA, "graph instantiate failed: %s", cudaGetErrorString(e)); }
            s->graph_steps = G;
        }
        while (n_steps - done >= G) {
            SPIN_CUDA(cudaGraphLaunch(gexec, s->stream));
            s->n_launch += s->graph_launches;
            done += G;
        }
    }
    const int64_t rest = n_steps - done;
    for (int64_t k = 0; k < rest; ++k) {
        rc = enqueue_step(s, (unsigned)k);
        if (rc) return rc;
    }
    if (rest > 0) {
        advance_step_kernel<<<1, 1, 0, s->stream>>>(s->d_step, (unsigned long long)rest);
        s->n_launch++;
    }
    s->step += (uint64_t)n_steps;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

// ---------------------------------------------------------------------------------------------- slab decomposition along c
// Several GPUs share one lattice: each holds a slab of planes and the ghost layers along c are filled by a halo exchange before every
// sweep.  The library provides the pieces -- the ghost-aware plan, sweeps over brick ranges, the halo
// planes as contiguous device chunks; the driver (paper_1901_11350_b200/slab.py) orders them and owns the transport (NCCL / peer copies).
extern "C" int spin_set_slab(spin_system *s, int enabled, int c_offset, int global_cells_c, int global_periodic_c) {
    REQUIRE(s, "null system");
    if (!enabled) { s->slab_on = 0; s->slab_off = 0; s->slab_gnc = 0; s->slab_gper = 0; s->plan_dirty = true; drop_graphs(s); return SPIN_OK; }
    REQUIRE(global_cells_c >= s->nc[2] && c_offset >= 0 && c_offset + s->nc[2] <= global_cells_c, "slab [%d, %d) does not lie inside %d planes", c_offset,
            c_offset + s->nc[2], global_cells_c);
    REQUIRE(s->n_img == 1, "slab decomposition and batched images are separate axes of parallelism");
    s->slab_on = 1; s->slab_off = c_offset; s->slab_gnc = global_cells_c; s->slab_gper = global_periodic_c ? 1 : 0;
    s->plan_dirty = true;
    drop_graphs(s);
    return SPIN_OK;
}
namespace {
// the per-spin array a halo call addresses: 0 the current configuration n, 1 the predictor n^p, 2 the next configuration (corrector output)
double *slab_array(spin_system *s, int array) { return array == 0 ? s->d_n[s->cur] : (array == 1 ? s->d_np : s->d_n[s->cur ^ 1]); }
int slab_ready(spin_system *s) {
    int rc = ensure_plan(s);
    if (rc) return rc;
    if (!s->slab_on) return spin::fail(SPIN_ERR_STATE, "not a slab: call spin_set_slab first");
    if (!jit_ready(s)) return spin::fail(SPIN_ERR_STATE, "slab sweeps need the run-time specialised kernels (%s)", s->jit_note.c_str());
    if (s->solver == SPIN_SOLVER_RK4) return spin::fail(SPIN_ERR_STATE, "slab sweeps are the two-stage solvers (Depondt, Heun, SIB)");
    return SPIN_OK;
}
}  // namespace
// doubles one side of the halo holds: reach along c x padded plane (ghost rows and columns included: they carry the in-plane images) x sublattices
extern "C" int spin_halo_doubles(spin_system *s, int64_t *doubles_per_side, int *reach_c) {
    REQUIRE(s && doubles_per_side, "null argument");
    int rc = slab_ready(s);
    if (rc) return rc;
    *doubles_per_side = (int64_t)s->nb * s->plan.rC * 3 * s->plan.PA * s->plan.PB;
    if (reach_c) *reach_c = s->plan.rC;
    return SPIN_OK;
}
// side 0 / 1 = towards lower / higher c.  get: the rC outermost OWN planes on that side -> dst (device, contiguous, sublattice-major);
// put: src -> the rC GHOST planes on that side.  Copies are enqueued on `stream` (NULL: the system's stream); nothing is synchronised.
extern "C" int spin_halo_get(spin_system *s, int array, int side, double *dst_device, void *stream) {
    REQUIRE(s && dst_device && array >= 0 && array <= 2 && (side == 0 || side == 1), "bad argument");
    int rc = slab_ready(s);
    if (rc) return rc;
    const DevicePlan &P = s->plan;
    const size_t plane = (size_t)3 * P.PA * P.PB, chunk = plane * P.rC;
    const size_t first = (size_t)(side == 0 ? P.LC : P.LC + P.Nc - P.rC) * plane;
    cudaStream_t st = stream ? (cudaStream_t)stream : s->stream;
    for (int b = 0; b < s->nb; ++b)
        SPIN_CUDA(cudaMemcpyAsync(dst_device + (size_t)b * chunk, slab_array(s, array) + (size_t)b * P.sub + first, chunk * sizeof(double), cudaMemcpyDeviceToDevice, st));
    return SPIN_OK;
}
extern "C" int spin_halo_put(spin_system *s, int array, int side, const double *src_device, void *stream) {
    REQUIRE(s && src_device && array >= 0 && array <= 2 && (side == 0 || side == 1), "bad argument");
    int rc = slab_ready(s);
    if (rc) return rc;
    const DevicePlan &P = s->plan;
    const size_t plane = (size_t)3 * P.PA * P.PB, chunk = plane * P.rC;
    const size_t first = (size_t)(side == 0 ? P.LC - P.rC : P.LC + P.Nc) * plane;
    cudaStream_t st = stream ? (cudaStream_t)stream : s->stream;
    for (int b = 0; b < s->nb; ++b)
        SPIN_CUDA(cudaMemcpyAsync(slab_array(s, array) + (size_t)b * P.sub + first, src_device + (size_t)b * chunk, chunk * sizeof(double), cudaMemcpyDeviceToDevice, st));
    return SPIN_OK;
}
// One sweep of the current step over part of the slab: stage 0 predictor (n -> n^p), 1 corrector (n, n^p -> next n);
// part 0 every brick, 1 the brick layers that hold planes a neighbour needs (within the reach of either face), 2 the layers in between.
// The driver launches part 1, starts the halo copies of its output, and launches part 2 while they travel.
extern "C" int llg_slab_sweep(spin_system *s, int stage, int part) {
    REQUIRE(s && (stage == 0 || stage == 1) && part >= 0 && part <= 2, "bad argument");
    int rc = slab_ready(s);
    if (rc) return rc;
    s->vp_active = false;
    const DevicePlan &P = s->plan;
    int b[3];
    jit_brick_shape(s, b);
    const int per_layer = ((P.Na + b[0] - 1) / b[0]) * ((P.Nb + b[1] - 1) / b[1]), layers = (P.Nc + b[2] - 1) / b[2];
    const int lo_end = std::min(layers, (P.rC + b[2] - 1) / b[2]), hi_begin = std::max(lo_end, (P.Nc - P.rC) / b[2]);      // boundary layers: [0, lo_end) and [hi_begin, layers)
    int ranges[2][2] = {{0, 0}, {0, 0}};
    if (part == 0) { ranges[0][0] = 0; ranges[0][1] = layers; }
    else if (part == 1) { ranges[0][0] = 0; ranges[0][1] = lo_end; ranges[1][0] = hi_begin; ranges[1][1] = layers; }
    else { ranges[0][0] = lo_end; ranges[0][1] = hi_begin; }
    double *n = s->d_n[s->cur], *nout = s->d_n[s->cur ^ 1];
    const Launch L = brick_launch(s);
    for (int r = 0; r < 2; ++r) {
        const int nl = ranges[r][1] - ranges[r][0];
        if (nl <= 0) continue;
        const unsigned brick0 = (unsigned)(ranges[r][0] * per_layer), count = (unsigned)(nl * per_layer);
        rc = stage == 0 ? jit_launch_predictor(s, L.grid, L.block, n, s->d_fddi[0], s->d_np, s->d_A, 0u, brick0, count)
                        : jit_launch_corrector(s, L.grid, L.block, n, s->d_np, s->d_fddi[0], s->d_fddi[1], s->d_A, nout, 0u, brick0, count);
        if (rc) return rc;
        s->n_launch++;
    }
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
// The whole Depondt step of a slab in one pass (the plane-marching kernel; spin_kernel_info says "jit+march"): reads the current
// configuration with ghost layers of depth 2 x reach along c (spin_halo_doubles reports that depth), writes the next configuration's own
// planes.  The driver then exchanges the halos of the next configuration (array 2) ONCE and calls llg_slab_advance.  part 0: the whole
// slab; 1: the first and the last chunk of planes (they hold what the neighbours need); 2: the chunks in between, which run while the halos travel.
extern "C" int llg_slab_step(spin_system *s, int part) {
    REQUIRE(s && part >= 0 && part <= 2, "bad argument");
    int rc = slab_ready(s);
    if (rc) return rc;
    if (!jit_march_ready(s)) return spin::fail(SPIN_ERR_STATE, "llg_slab_step needs the one-pass marching kernel (spin_kernel_info: %s); use llg_slab_sweep", "not jit+march");
    s->vp_active = false;
    rc = jit_launch_march(s, s->cur, s->d_n[s->cur ^ 1], 0u, part);
    if (rc) return rc;
    if (part == 0) s->n_launch++;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
// The same step with the halo exchange FUSED into the kernel: the boundary planes of the next configuration are written by the kernel
// itself into the neighbours' ghost layers (peer_lo_next / peer_hi_next: the neighbours' next-configuration arrays from spin_slab_arrays,
// device pointers this GPU can write -- peer access over NVLink, an opened IPC handle, or another system of this device; NULL at an open
// end).  No halo copy and no message follow; what remains for the driver is ORDER: this call must come after both neighbours' previous
// step has completed (they wrote this slab's ghost layers and read the arrays this step overwrites), e.g. by stream waits on their events.
extern "C" int llg_slab_step_fused(spin_system *s, double *peer_lo_next, int peer_lo_cells_c, double *peer_hi_next) {
    REQUIRE(s, "null system");
    int rc = slab_ready(s);
    if (rc) return rc;
    if (!jit_march_ready(s)) return spin::fail(SPIN_ERR_STATE, "llg_slab_step_fused needs the one-pass marching kernel (spin_kernel_info: %s); use llg_slab_sweep", "not jit+march");
    REQUIRE(!peer_lo_next || peer_lo_cells_c >= s->plan.rC, "lower neighbour thinner than the ghost depth");
    s->vp_active = false;
    rc = jit_launch_march(s, s->cur, s->d_n[s->cur ^ 1], 0u, 0, peer_lo_next, peer_hi_next, peer_lo_cells_c);
    if (rc) return rc;
    s->n_launch++;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
// device pointers of the current and the next configuration array (padded layout of DESIGN.md section 2, ghost layers included): what a
// neighbouring slab writes into (llg_slab_step_fused).  They swap roles at every llg_slab_advance.
extern "C" int spin_slab_arrays(spin_system *s, double **current, double **next) {
    REQUIRE(s && current && next, "null argument");
    int rc = slab_ready(s);
    if (rc) return rc;
    *current = s->d_n[s->cur]; *next = s->d_n[s->cur ^ 1];
    return SPIN_OK;
}
// ---- between PROCESSES (one per GPU): the neighbours' arrays are mapped through CUDA IPC and the order of the steps is kept by flags in
// device memory instead of events (an event of another process cannot say WHICH record a wait refers to): after its step k a slab writes
// k into a flag of each neighbour (release, system scope, stream-ordered after the step's kernel); before its step k + 1 it waits until
// both its flags hold k.  The wait is a one-thread kernel that polls with a bound and traps when the bound is hit (a lost neighbour ends
// the launch with an error, never hangs the device).  Each kernel waits on ANOTHER GPU's progress: never run two such ranks on one GPU.
namespace {
__global__ void flag_signal_kernel(unsigned long long *flag, unsigned long long value) {
    asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(flag), "l"(value) : "memory");
}
__global__ void flag_wait_kernel(const unsigned long long *flag, unsigned long long value) {
    unsigned long long v = 0, t0 = 0, t = 0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (;;) {
        asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(flag) : "memory");
        if (v >= value) return;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (t - t0 > 30000000000ull) __trap();      // 30 s without the neighbour: an error, not a hang
    }
}
}  // namespace
extern "C" int spin_slab_flags(spin_system *s, unsigned long long **flags) {
    REQUIRE(s && flags, "null argument");
    NEED_DEVICE(s);
    if (!s->d_flags) {
        SPIN_CUDA(cudaMalloc(&s->d_flags, 2 * sizeof(unsigned long long)));
        SPIN_CUDA(cudaMemsetAsync(s->d_flags, 0, 2 * sizeof(unsigned long long), s->stream));
        // both kernels run once now: the first launch of a kernel may load its module, which cannot happen while a wait is polling
        flag_signal_kernel<<<1, 1, 0, s->stream>>>(s->d_flags, 0ull);
        flag_wait_kernel<<<1, 1, 0, s->stream>>>(s->d_flags, 0ull);
        SPIN_CUDA(cudaStreamSynchronize(s->stream));
    }
    *flags = s->d_flags;
    return SPIN_OK;
}
extern "C" int spin_flag_signal(spin_system *s, unsigned long long *flag, unsigned long long value) {
    REQUIRE(s && flag, "null argument");
    NEED_DEVICE(s);
    flag_signal_kernel<<<1, 1, 0, s->stream>>>(flag, value);
    s->n_launch++;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
extern "C" int spin_flag_wait(spin_system *s, const unsigned long long *flag, unsigned long long value) {
    REQUIRE(s && flag, "null argument");
    NEED_DEVICE(s);
    flag_wait_kernel<<<1, 1, 0, s->stream>>>(flag, value);
    s->n_launch++;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
// CUDA IPC: the handle of the ALLOCATION that holds `device_ptr` and the pointer's offset inside it (small allocations share one), to be
// sent to the neighbour's process by any means; spin_ipc_open maps it there and returns the same address plus offset
extern "C" int spin_ipc_export(const void *device_ptr, unsigned char handle[64], int64_t *offset) {
    REQUIRE(device_ptr && handle && offset, "null argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handles are 64 bytes");
    typedef int (*range_fn)(unsigned long long *, size_t *, unsigned long long);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    SPIN_CUDA(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return spin::fail(SPIN_ERR_CUDA, "cuMemGetAddressRange is not available from this driver");
    unsigned long long base = 0;
    size_t size = 0;
    const int r = ((range_fn)fn)(&base, &size, (unsigned long long)(uintptr_t)device_ptr);
    if (r != 0) return spin::fail(SPIN_ERR_CUDA, "cuMemGetAddressRange failed: driver error %d", r);
    cudaIpcMemHandle_t h;
    SPIN_CUDA(cudaIpcGetMemHandle(&h, (void *)(uintptr_t)base));
    memcpy(handle, &h, 64);
    *offset = (int64_t)((unsigned long long)(uintptr_t)device_ptr - base);
    return SPIN_OK;
}
extern "C" int spin_ipc_open(const unsigned char handle[64], int64_t offset, void **device_ptr) {
    REQUIRE(handle && device_ptr && offset >= 0, "bad argument");
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    void *base = nullptr;
    SPIN_CUDA(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    *device_ptr = (char *)base + offset;
    return SPIN_OK;
}
extern "C" int spin_ipc_close(void *device_ptr, int64_t offset) {
    REQUIRE(device_ptr && offset >= 0, "bad argument");
    SPIN_CUDA(cudaIpcCloseMemHandle((char *)device_ptr - offset));
    return SPIN_OK;
}
// after the corrector sweeps of a step: the next configuration becomes the current one and the step counter (the noise stream) advances
extern "C" int llg_slab_advance(spin_system *s) {
    REQUIRE(s, "null system");
    int rc = slab_ready(s);
    if (rc) return rc;
    s->cur ^= 1;
    advance_step_kernel<<<1, 1, 0, s->stream>>>(s->d_step, 1ull);
    s->n_launch++;
    s->step += 1;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

extern "C" int spin_synchronize(spin_system *s) {
    REQUIRE(s, "null system");
    NEED_DEVICE(s);
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

// ---------------------------------------------------------------------------------------------- observables
extern "C" int effective_field_device(spin_system *s, double *B) {
    REQUIRE(s && B, "null argument");
    int rc = ensure_plan(s);
    if (rc) return rc;
    rc = enqueue_force(s, T_ALL, s->d_np);
    if (rc) return rc;
    // B = F / (mu_b mu_B), boundary order
    const int nt = 256;
    unpack_kernel<<<(unsigned)((s->N + nt - 1) / nt), nt, 0, s->stream>>>(s->plan, s->d_np, B, (int)s->N, 1);
    s->n_launch++;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
extern "C" int effective_field(spin_system *s, double *B) {
    REQUIRE(s && B, "null argument");
    int rc = effective_field_device(s, s->d_aos);
    if (rc) return rc;
    SPIN_CUDA(cudaMemcpyAsync(B, s->d_aos, (size_t)3 * s->N * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    SPIN_CUDA(cudaStreamSynchronize(s->stream));
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
extern "C" int energy(spin_system *s, double *E_total, double E_terms[6]) {
    REQUIRE(s, "null system");
    int rc = ensure_plan(s);
    if (rc) return rc;
    double r[N_RED];
    rc = reduce_all(s, r);
    if (rc) return rc;
    double tot = 0.0;
    for (int k = 0; k < 6; ++k) { if (E_terms) E_terms[k] = r[k]; tot += r[k]; }
    if (E_total) *E_total = tot;
    return SPIN_OK;
}
extern "C" int observables(spin_system *s, double M[3], double *max_torque) {
    REQUIRE(s, "null system");
    int rc = ensure_plan(s);
    if (rc) return rc;
    double r[N_RED];
    rc = reduce_all(s, r);
    if (rc) return rc;
    if (M) for (int k = 0; k < 3; ++k) M[k] = r[6 + k] / (double)s->N;
    if (max_torque) *max_torque = r[9];
    return SPIN_OK;
}

// Velocity-projection minimiser (App. D): 3 own launches per iteration (+ the dipolar field)
extern "C" int minimise_vp(spin_system *s, int64_t n_iter, double dt, double mass) {
    REQUIRE(s && n_iter >= 0, "bad argument");
    REQUIRE(dt > 0.0 && isfinite(dt) && mass > 0.0 && isfinite(mass), "dt and mass must be positive");
    if (s->n_img > 1) return spin::fail(SPIN_ERR_STATE, "minimise_vp works on a single image");
    int rc = ensure_plan(s);
    if (rc) return rc;
    const Launch L = brick_launch(s);
    const int nblocks = (int)(L.grid.x * L.grid.y);
    double *Fbuf[2] = {s->d_A, s->d_fddi[1]};
    if (!s->vp_active) {
        SPIN_CUDA(cudaMemsetAsync(s->d_vp, 0, 4 * sizeof(double), s->stream));
        SPIN_CUDA(cudaMemsetAsync(Fbuf[0], 0, (size_t)s->nb * s->plan.sub * sizeof(double), s->stream));
        s->vp_cur = 0;
        s->vp_active = true;
    }
    double *n = s->d_n[s->cur];
    const double c = 0.5 * dt / mass, h = 0.5 * dt * dt / mass;
    for (int64_t it = 0; it < n_iter; ++it) {
        if (s->ddi_on) { rc = ddi_field(s, n, s->d_fddi[0]); if (rc) return rc; }
        double *Fold = Fbuf[s->vp_cur], *Fnew = Fbuf[s->vp_cur ^ 1];
        if (L.flat) vp_force_kernel<32, 8, 1><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], Fold, Fnew, s->d_partials);
        else vp_force_kernel<32, 4, 2><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, s->d_fddi[0], Fold, Fnew, s->d_partials);
        vp_final_kernel<<<1, 32, 0, s->stream>>>(s->d_partials, nblocks, c, s->d_vp);
        if (L.flat) vp_update_kernel<32, 8, 1><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, Fnew, s->d_vp, dt, h);
        else vp_update_kernel<32, 4, 2><<<L.grid, L.block, 0, s->stream>>>(s->plan, n, Fnew, s->d_vp, dt, h);
        s->n_launch += 3;
        s->vp_cur ^= 1;
    }
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}
extern "C" int minimise_vp_reset(spin_system *s) {
    REQUIRE(s, "null system");
    s->vp_active = false;
    return SPIN_OK;
}

// ---- GNEB on the batched images (III.D, App. F): images 0 and n_img-1 are the fixed ends of the chain
namespace {
int gneb_run(spin_system *s, int64_t n_iter, double step, double kappa, int climbing, bool want_outputs, double *F_host, double *E_host, double *l_host) {
    const int M = s->n_img;
    const Launch L = brick_launch(s);
    const int nblocks = (int)(L.grid.x * L.grid.y);
    const size_t istr = (size_t)s->nb * s->plan.sub;
    // one scratch block (nothing to leak on an error path): partial sums, per-image scalars, energies, N_RED reductions per image (the
    // energies never leave the device during the relaxation)
    double *d_scratch = nullptr;
    const size_t n_part = (size_t)M * nblocks * 3, n_sc = (size_t)M * 3, n_E = (size_t)M, n_red = (size_t)M * 16;
    SPIN_CUDA(cudaMalloc(&d_scratch, (n_part + n_sc + n_E + n_red) * sizeof(double)));
    double *d_part = d_scratch, *d_sc = d_part + n_part, *d_E = d_sc + n_sc, *d_red = d_E + n_E;
    const int sel = s->img_sel;
    int rc = SPIN_OK;
    dim3 grid(L.grid.x, L.grid.y, (unsigned)M);
    double *n_all = s->d_n[s->cur], *G_all = s->d_np, *tau_all = s->d_A;
    for (int64_t it = 0; it < n_iter && rc == SPIN_OK; ++it) {
        for (int nu = 0; nu < M && rc == SPIN_OK; ++nu) {          // energy and force of every image
            s->img_sel = nu;
            rc = enqueue_reduce(s, d_red + 16 * nu);
            if (rc == SPIN_OK) rc = enqueue_force(s, T_ALL, G_all + nu * istr);
        }
        if (rc) break;
        gneb_energy_kernel<<<1, 64, 0, s->stream>>>(d_red, M, d_E);
        s->n_launch++;
        const double st = want_outputs ? 0.0 : step;
        if (L.flat) {
            gneb_tangent_kernel<32, 8, 1><<<grid, L.block, 0, s->stream>>>(s->plan, n_all, G_all, d_E, M, istr, tau_all, d_part);
            gneb_final_kernel<<<M, 32, 0, s->stream>>>(d_part, nblocks, d_sc);
            gneb_assemble_kernel<32, 8, 1><<<grid, L.block, 0, s->stream>>>(s->plan, n_all, G_all, tau_all, d_sc, M, istr, kappa, climbing, st);
        } else {
            gneb_tangent_kernel<32, 4, 2><<<grid, L.block, 0, s->stream>>>(s->plan, n_all, G_all, d_E, M, istr, tau_all, d_part);
            gneb_final_kernel<<<M, 32, 0, s->stream>>>(d_part, nblocks, d_sc);
            gneb_assemble_kernel<32, 4, 2><<<grid, L.block, 0, s->stream>>>(s->plan, n_all, G_all, tau_all, d_sc, M, istr, kappa, climbing, st);
        }
        s->n_launch += 3;
    }
    if (rc == SPIN_OK) {
        cudaError_t e = cudaStreamSynchronize(s->stream);
        if (e != cudaSuccess) rc = spin::fail(SPIN_ERR_CUDA, "gneb: %s", cudaGetErrorString(e));
    }
    if (rc == SPIN_OK && want_outputs) {
        if (E_host) { cudaMemcpyAsync(E_host, d_E, (size_t)M * sizeof(double), cudaMemcpyDeviceToHost, s->stream); cudaStreamSynchronize(s->stream); }
        if (l_host) {
            std::vector<double> sc((size_t)3 * M);
            cudaMemcpyAsync(sc.data(), d_sc, sc.size() * sizeof(double), cudaMemcpyDeviceToHost, s->stream);
            cudaStreamSynchronize(s->stream);
            for (int nu = 0; nu < M; ++nu) l_host[nu] = sc[(size_t)3 * nu + 2];
        }
        if (F_host) {
            const int nt = 256;
            for (int nu = 0; nu < M; ++nu) {
                unpack_kernel<<<(unsigned)((s->N + nt - 1) / nt), nt, 0, s->stream>>>(s->plan, G_all + nu * istr, s->d_aos, (int)s->N, 0);
                s->n_launch++;
                cudaMemcpyAsync(F_host + (size_t)nu * 3 * s->N, s->d_aos, (size_t)3 * s->N * sizeof(double), cudaMemcpyDeviceToHost, s->stream);
                cudaStreamSynchronize(s->stream);
            }
        }
    }
    s->img_sel = sel;
    cudaFree(d_scratch);
    if (rc == SPIN_OK && cudaGetLastError() != cudaSuccess) rc = spin::fail(SPIN_ERR_CUDA, "gneb: kernel launch failed");
    return rc;
}
}  // namespace

extern "C" int gneb_forces(spin_system *s, double kappa, int climbing_image, double *F_xyz, double *E_meV, double *l_geodesic) {
    REQUIRE(s, "null system");
    REQUIRE(s->n_img >= 3, "a chain needs at least 3 images (spin_set_images)");
    REQUIRE(climbing_image < s->n_img, "climbing image out of range");
    int rc = ensure_plan(s);
    if (rc) return rc;
    s->vp_active = false;
    return gneb_run(s, 1, 0.0, kappa, climbing_image, true, F_xyz, E_meV, l_geodesic);
}
extern "C" int gneb_iterate(spin_system *s, int64_t n_iterations, double step, double kappa, int climbing_image) {
    REQUIRE(s && n_iterations >= 0 && step > 0.0 && isfinite(step), "bad argument");
    REQUIRE(s->n_img >= 3, "a chain needs at least 3 images (spin_set_images)");
    REQUIRE(climbing_image < s->n_img, "climbing image out of range");
    int rc = ensure_plan(s);
    if (rc) return rc;
    s->vp_active = false;
    return gneb_run(s, n_iterations, step, kappa, climbing_image, false, nullptr, nullptr, nullptr);
}

// Q of App. A summed over the a-b planes; one basis atom
extern "C" int topological_charge(spin_system *s, double *Q) {
    REQUIRE(s && Q, "null argument");
    REQUIRE(s->nb == 1, "the topological charge is defined for one basis atom (triangulation of a Bravais lattice)");
    int rc = ensure_plan(s);
    if (rc) return rc;
    const int nblk = (int)((s->ncell + 255) / 256);
    const int ccw = (s->brav[0] * s->brav[4] - s->brav[1] * s->brav[3]) > 0.0 ? 1 : 0;
    double *d_part = nullptr;
    SPIN_CUDA(cudaMalloc(&d_part, (size_t)nblk * sizeof(double)));
    topo_kernel<<<nblk, 256, 0, s->stream>>>(s->plan, s->d_n[s->cur] + img_off(s), ccw, d_part);
    topo_final_kernel<<<1, 32, 0, s->stream>>>(d_part, nblk, s->d_result);
    s->n_launch += 2;
    cudaError_t e = cudaMemcpyAsync(Q, s->d_result, sizeof(double), cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    cudaFree(d_part);
    if (e != cudaSuccess) return spin::fail(SPIN_ERR_CUDA, "topological_charge: %s", cudaGetErrorString(e));
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

// The same reduction for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
// the per-block partial sums live in a file-scope device array instead of a buffer allocated per call.  Every GPU that loads the library
// holds the array (128 KB) until exit.  In host code the array's NAME is a host-side stand-in, not a device address: the address is resolved
// with cudaGetSymbolAddress at set-up (spin_system_create), once per device with that device current, and that pointer goes to the kernels.
constexpr int TOPO_NOALLOC_MAX_BLOCKS = 16384;                         // x 256 cells per block = 4,194,304 cells
constexpr int TOPO_NOALLOC_MAX_DEVICES = 64;
static __device__ __align__(256) double g_topo_scratch[TOPO_NOALLOC_MAX_BLOCKS];
static double *g_topo_scratch_addr[TOPO_NOALLOC_MAX_DEVICES];          // device address of g_topo_scratch, per device; nullptr: not resolved
static std::mutex g_topo_mutex;

static int topo_noalloc_setup() {
    int dev = -1;
    SPIN_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= TOPO_NOALLOC_MAX_DEVICES) return spin::fail(SPIN_ERR_LIMIT, "device ordinal %d beyond the %d this library keeps scratch addresses for", dev, TOPO_NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_topo_mutex);
    if (g_topo_scratch_addr[dev]) return SPIN_OK;
    double *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_topo_scratch);
    if (e != cudaSuccess || !ptr) return spin::fail(SPIN_ERR_CUDA, "cudaGetSymbolAddress(g_topo_scratch) on device %d: %s", dev, cudaGetErrorString(e));
    g_topo_scratch_addr[dev] = ptr;
    return SPIN_OK;
}

extern "C" int topological_charge_noalloc(spin_system *s, double *d_Q) {
    REQUIRE(s && d_Q, "null argument");
    NEED_DEVICE(s);
    REQUIRE(s->nb == 1, "the topological charge is defined for one basis atom (triangulation of a Bravais lattice)");
    const int64_t nblk = (s->ncell + 255) / 256;
    if (nblk > TOPO_NOALLOC_MAX_BLOCKS)
        return spin::fail(SPIN_ERR_LIMIT, "topological_charge_noalloc: %lld cells exceed the fixed scratch array (%d blocks of 256 cells = %lld cells); use topological_charge",
                          (long long)s->ncell, TOPO_NOALLOC_MAX_BLOCKS, (long long)TOPO_NOALLOC_MAX_BLOCKS * 256);
    if (s->plan_dirty)
        return spin::fail(SPIN_ERR_STATE, "topological_charge_noalloc: the plan is not built and building it allocates; call spins_set, effective_field, "
                                          "topological_charge or llg_iterate once after the last change of the lattice, Hamiltonian or options");
    int dev = -1;
    SPIN_CUDA(cudaGetDevice(&dev));
    double *scratch = (dev >= 0 && dev < TOPO_NOALLOC_MAX_DEVICES) ? g_topo_scratch_addr[dev] : nullptr;
    if (!scratch) return spin::fail(SPIN_ERR_STATE, "topological_charge_noalloc: no scratch address for device %d (create the system with this device current)", dev);
    const int ccw = (s->brav[0] * s->brav[4] - s->brav[1] * s->brav[3]) > 0.0 ? 1 : 0;
    // every block overwrites its own partial sum and the final kernel reads the first nblk only: nothing has to start at zero
    topo_kernel<<<(unsigned)nblk, 256, 0, s->stream>>>(s->plan, s->d_n[s->cur] + img_off(s), ccw, scratch);
    topo_final_kernel<<<1, 32, 0, s->stream>>>(scratch, (int)nblk, d_Q);
    s->n_launch += 2;
    SPIN_CUDA(cudaGetLastError());
    return SPIN_OK;
}

// ---------------------------------------------------------------------------------------------- introspection
extern "C" int spin_launch_counts(const spin_system *s, int64_t *own, int64_t *fft) {
    REQUIRE(s, "null system");
    if (own) *own = s->n_launch;
    if (fft) *fft = s->n_fft;
    return SPIN_OK;
}
// measured fp64 FMA throughput of the device in TFLOP/s (2 flops per fma), best of 5 launches of a register-only kernel
extern "C" int spin_measure_fp64_tflops(spin_system *s, double *tflops) {
    REQUIRE(s && tflops, "null argument");
    NEED_DEVICE(s);
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int iters = 1 << 14, blocks = sms * 16;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        SPIN_CUDA(cudaEventRecord(s->ev0, s->stream));
        fp64_rate_kernel<<<blocks, 256, 0, s->stream>>>(s->d_result, iters, 0.999999, 1e-9);
        SPIN_CUDA(cudaEventRecord(s->ev1, s->stream));
        SPIN_CUDA(cudaEventSynchronize(s->ev1));
        float ms = 0.f;
        SPIN_CUDA(cudaEventElapsedTime(&ms, s->ev0, s->ev1));
        const double tf = 2.0 * 8.0 * (double)iters * 256.0 * blocks / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    s->n_launch += 6;
    *tflops = best;
    return SPIN_OK;
}
extern "C" int spin_profile_enable(spin_system *s, int on) {
    REQUIRE(s, "null system");
    s->profile_on = on ? 1 : 0;
    for (int k = 0; k < 3; ++k) { s->prof_ms[k] = 0; s->prof_n[k] = 0; }
    return SPIN_OK;
}
extern "C" int spin_profile_get(spin_system *s, int kind, double *ms, int64_t *n) {
    REQUIRE(s && kind >= 0 && kind < 4, "bad argument");
    if (ms) *ms = s->prof_ms[kind];
    if (n) *n = s->prof_n[kind];
    return SPIN_OK;
}
extern "C" int spin_set_option(spin_system *s, const char *name, int value) {
    REQUIRE(s && name, "null argument");
    if (!strcmp(name, "use_graph")) s->opt_graph = value ? 1 : 0;
    else if (!strcmp(name, "store_A")) { s->opt_store_A = value ? 1 : 0; s->plan_dirty = true; }
    else if (!strcmp(name, "use_jit")) { s->opt_jit = value ? 1 : 0; s->plan_dirty = true; }
    else if (!strcmp(name, "use_coop")) { s->opt_coop = value < 0 ? 0 : (value > 3 ? 3 : value); s->plan_dirty = true; }
    else if (!strcmp(name, "cache_noise")) { s->opt_cache_noise = value ? 1 : 0; s->plan_dirty = true; }
    else if (!strcmp(name, "use_pdl")) { s->opt_pdl = value > 2 ? -1 : value < 0 ? -1 : value; s->plan_dirty = true; }
    else if (!strcmp(name, "use_march")) { s->opt_march = value < 0 ? 0 : (value > 2 ? 2 : value); s->plan_dirty = true; }
    else if (!strcmp(name, "ddi_mirror")) { s->opt_ddi_mirror = value ? 1 : 0; s->plan_dirty = true; }
    else if (!strcmp(name, "ddi_slab")) { s->opt_ddi_slab = value < 0 ? 0 : (value > 3 ? 3 : value); s->plan_dirty = true; }      // 0: 3-D path, 1: slab path, 2: slab path with cuFFT's a-pass, 3: own a-pass, cuFFT b-pass + separate contraction
    else return spin::fail(SPIN_ERR_ARG, "unknown option '%s'", name);
    drop_graphs(s);
    return SPIN_OK;
}

// which sweep kernels are in use: "jit" (run-time specialised) or "generic: <reason>"
extern "C" int spin_kernel_info(spin_system *s, char *buf, int len) {
    REQUIRE(s && buf && len > 0, "bad argument");
    if (s->has_device) { int rc = ensure_plan(s); if (rc) return rc; }
    if (jit_march_ready(s)) snprintf(buf, (size_t)len, "jit+march");
    else if (jit_coop_ready(s) && s->opt_coop && !s->ddi_on && (s->N <= SPIN_COOP_MAX_SPINS || s->opt_coop >= 2)) snprintf(buf, (size_t)len, jit_cluster_ready(s) ? "jit+cluster" : "jit+coop");
    else if (jit_ready(s)) snprintf(buf, (size_t)len, "jit (brick sweeps)");
    else snprintf(buf, (size_t)len, "generic: %s", s->jit_note.c_str());
    return SPIN_OK;
}
extern "C" int spin_ddi_info(spin_system *s, char *buf, int len) {
    REQUIRE(s && buf && len > 0, "bad argument");
    if (s->has_device) { int rc = ensure_plan(s); if (rc) return rc; }
    snprintf(buf, (size_t)len, "%s", ddi_path_name(s));
    return SPIN_OK;
}
extern "C" int spin_jit_compiler_info(char *buf, int len) {
    REQUIRE(buf && len > 0, "bad argument");
    snprintf(buf, (size_t)len, "%s", jit_compiler_info().c_str());
    return SPIN_OK;
}
// the generated translation unit of the specialised sweeps; with compile != 0 it is also compiled with NVRTC (no device
// needed) and the size of the cubin is returned in *cubin_bytes
extern "C" int spin_jit_source(spin_system *s, char *buf, int len, int compile, int64_t *cubin_bytes) {
    REQUIRE(s, "null system");
    int rc;
    if (s->has_device) {
        // a live system: bring plan, arrays and kernels up to date together (the plan must never describe a layout the arrays do not have)
        rc = ensure_plan(s);
        if (rc) return rc;
    } else {
        // planner-only mode: there are no device arrays; a plan that fails half-way must not replace the last good one
        DevicePlan P;
        rc = build_plan(s, P);
        if (rc) return rc;
        s->plan = P;
    }
    const std::string src = jit_source(s);
    if (buf && len > 0) snprintf(buf, (size_t)len, "%s", src.c_str());
    if (compile) {
        std::string cubin, log;
        rc = jit_compile(src, cubin, log);
        if (rc) return rc;
        if (cubin_bytes) *cubin_bytes = (int64_t)cubin.size();
    }
    return SPIN_OK;
}
