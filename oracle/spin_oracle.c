/*
 * spin_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU implementation of the hot path of "Spirit: Multifunctional
 * Framework for Atomistic Spin Simulations" (arXiv 1901.11350), written from the
 * paper's equations only.  It shares no code, header, table or constant generator
 * with the CUDA library under paper_1901_11350_b200/; only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call it.
 *
 * What it follows (PAPER.md line numbers):
 *   energy            Eq. 1 (:61-67), Eq. 2 (:75)           -> orc_energy
 *   gradient F=-dH/dn ":155  B_eff = -dH/dn_i"              -> orc_gradient (gather), orc_gradient_scatter
 *   dipole-dipole     :81-89 direct sum / FFT convolution   -> orc_ddi_direct, orc_ddi_fft
 *   LLG explicit form Eq. 10 (:147-153)                     -> rot_field()
 *   thermal field     Eq. 11 (:157-160)                     -> orc_thermal_xi, sigma
 *   Depondt solver    App. B, B5-B7 (:369-380)              -> orc_llg_step (solver 0)
 *   Heun solver       App. B, B3-B4 (:355-367)              -> orc_llg_step (solver 1); orc_heun_step = the same written on its own (pin)
 *   GNEB forces       III.D Eqs. 14-17 (:193-216), App. F   -> orc_gneb_forces, orc_gneb_iterate, orc_geodesic_distance
 *   velocity projection App. D, D1-D5 (:438-463)            -> orc_vp_iterate
 *   topological charge App. A, A1-A2 (:317-343)             -> orc_topological_charge, orc_spherical_area
 *   RK4 solver        :168 (named only; textbook tableau)   -> orc_llg_step (solver 3), orc_rk4_step
 *   SIB solver        App. C, C5-C11 (:384-436)             -> orc_llg_step (solver 2), imp_update (Cramer's rule as printed)
 * Readings of silent / garbled passages are listed in DESIGN.md ("Readings") under the
 * same R-numbers as SURVEY.md 8(c).
 *
 * Units: energy meV, field T, moments mu_B, time ps, length Angstrom.
 * Spin index (same as the C-ABI boundary): i = b + n_basis*(ia + Na*(ib + Nb*ic)).
 * Spins are stored AoS: n[3*i + {0,1,2}].
 *
 * Parity pins (tests/test_oracle_pins.py): FM closed form, Larmor Eq. 12 with the paper's printed 3e-7 error, finite differences,
 * Euler identity, brute-force DDI, two-dipole and monolayer closed forms, spin-spiral closed form, Langevin <n_z>, Philox known
 * answers; Heun / SIB / RK4: convergence orders 2 / 2 / 4 on Eq. 12 and the exact Cayley rotation 2 atan(gamma B dt / 2); damping-only
 * dynamics: tanh at fixed azimuth; velocity projection: (k + 1/2) dt^2 F / m and the FM ground state; pinned spins: Eq. 12 about the
 * pinned neighbour; vacancies: decoupled neighbours; several anisotropy axes: biaxial closed form; topological charge: octant area,
 * Girard's excess, Q = -1 / +1 / 0 / -2; GNEB: geodesic distance, force geometry, equidistant relaxation, barrier = K with a climbing
 * image; image noise streams: moments and cross-correlations; current-driven wall of Fig. 6: velocity (beta / alpha) u;
 * orc_effective_field: free spins feel the applied field in Tesla for mu_s = 2 and 5, ferromagnet B + (2K + zJ)/(mu_s mu_B), per-atom
 * moments; orc_observables: M of a known configuration, max torque mu_s mu_B B sin(theta) of one tilted spin and |n x F| with a bond.
 * "parity unpinned" (convention only): DMI chirality sign of the helper conventions (R15), DDI image count (R16),
 * periodic self-wrap (R21), the choice of the max norm over spins for "max torque" (R22; its value is pinned), the optimiser of the
 * GNEB chain (steepest descent, R31).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA-2018 (paper is silent on constants, reading R5) */
#define ORC_MU_B   0.057883818060   /* meV / T            */
#define ORC_K_B    0.08617333262    /* meV / K            */
#define ORC_GAMMA  0.176085963023   /* rad / (ps T)       */
#define ORC_C_DD   0.0536815112     /* mu0 mu_B^2/(4 pi A^3), meV */
#define ORC_PI     3.14159265358979323846

enum { T_ZEE = 1, T_ANI = 2, T_EXC = 4, T_DMI = 8, T_QUAD = 16, T_DDI = 32, T_ALL = 63 };

typedef struct orc_system {
    double brav[9];          /* rows a, b, c in units of alat                      */
    int nb;                  /* atoms in the basis                                 */
    double *basis;           /* 3*nb fractional coordinates                        */
    int nc[3], per[3];       /* cells and periodic flags per direction             */
    double alat;             /* lattice constant, Angstrom                         */
    long ncell, N;
    double *mu;              /* nb, mu_B                                           */
    double *mu_site;         /* N moments in boundary order or NULL: ":79 atoms of different types" -- a per-site moment that
                                replaces the basis atom's wherever mu_i enters (Zeeman term and dipolar sum of Eq. 1, the 1/mu_i of
                                Eq. 10, the thermal amplitude of Eq. 11, the conversion of the boundary to Tesla); reading R32  */
    double Bext[3];          /* Tesla                                              */
    double *K, *Kax;         /* legacy single-axis view (first entry per atom); the sums run over the entry list below */
    int nani; int *ab; double *aK, *aax;   /* anisotropy entries: basis atom, K, unit axis -- "sum_i sum_j K_j (K^_j . n_i)^2" (Eq. 1 :61)
                                              has a sum over axes j: an atom may carry several (reading R3, extended)             */
    int npairs; int *pi, *pj, *pt; double *pJ, *pD;
    int nquads; int *qb, *qt; double *qK;
    int ddi, nimg[3];
    int ddi_direct;          /* 1: stepping/energy use the O(N^2) sum              */
    /* padded-FFT cache */
    int P[3]; long Ptot; double *Khat;   /* [a][b][6][Ptot] complex interleaved     */
    /* LLG */
    double dt, alpha, T, u, jdir[3], beta;
    uint64_t seed, step;
    double *n;               /* 3N */
    int nthreads;
    unsigned char *pinned;   /* N flags or NULL: a pinned spin keeps its value (":79 pinning of individual spins"); a vacancy
                                (":79 defects, such as vacancies") is a pinned site holding the zero vector (reading R27)   */
    double *vp_v, *vp_F;     /* velocity-projection minimiser (App. D): velocity and force of the previous iteration, or NULL  */
    uint32_t image;          /* which image's noise stream this system draws (0 = the single-system stream)                    */
    int damping_only;        /* 1: the precession term of Eq. 10 is dropped (:168), the solvers become minimisers                */
    int solver;              /* 0 Depondt (App. B B5-B7), 1 Heun (B3-B4), 2 SIB semi-implicit midpoint (App. C), 3 RK4 (:168) */
} orc_system;

/* moment of spin i (mu_B): its own if per-site moments are set, else its basis atom's (i = b + nb * cell) */
static inline double mu_at(const orc_system *s, long i) { return s->mu_site ? s->mu_site[i] : s->mu[i % s->nb]; }


/* ------------------------------------------------------------------ helpers */
static inline long cell_index(const orc_system *s, const int c[3]) {
    return c[0] + (long)s->nc[0] * (c[1] + (long)s->nc[1] * c[2]);
}
static inline void cell_coords(const orc_system *s, long cell, int c[3]) {
    c[0] = (int)(cell % s->nc[0]);
    c[1] = (int)((cell / s->nc[0]) % s->nc[1]);
    c[2] = (int)(cell / ((long)s->nc[0] * s->nc[1]));
}
/* cell c + sign*t with boundary conditions; returns 0 if it falls off an open edge
 * (reading R20), wraps modulo n_cells in periodic directions (reading R21).        */
static inline int shifted_cell(const orc_system *s, const int c[3], const int t[3], int sign, int out[3]) {
    for (int d = 0; d < 3; ++d) {
        int x = c[d] + sign * t[d];
        if (x < 0 || x >= s->nc[d]) {
            if (!s->per[d]) return 0;
            x %= s->nc[d];
            if (x < 0) x += s->nc[d];
        }
        out[d] = x;
    }
    return 1;
}
static inline long spin_index(const orc_system *s, const int c[3], int b) {
    return b + (long)s->nb * cell_index(s, c);
}
static inline double dot3(const double *a, const double *b) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static inline void cross3(const double *a, const double *b, double *o) {
    o[0] = a[1]*b[2] - a[2]*b[1];
    o[1] = a[2]*b[0] - a[0]*b[2];
    o[2] = a[0]*b[1] - a[1]*b[0];
}
/* Cartesian position (Angstrom) of fractional lattice coordinate f (cells + basis) */
static inline void frac_to_cart(const orc_system *s, const double f[3], double r[3]) {
    for (int k = 0; k < 3; ++k)
        r[k] = s->alat * (f[0]*s->brav[0+k] + f[1]*s->brav[3+k] + f[2]*s->brav[6+k]);
}

/* ------------------------------------------------------------------ lifecycle */
orc_system *orc_create(const double brav[9], int nb, const double *basis, const int nc[3],
                       const int per[3], double alat) {
    orc_system *s = (orc_system *)calloc(1, sizeof(orc_system));
    memcpy(s->brav, brav, 9 * sizeof(double));
    s->nb = nb;
    s->basis = (double *)malloc(3 * nb * sizeof(double));
    memcpy(s->basis, basis, 3 * nb * sizeof(double));
    for (int d = 0; d < 3; ++d) { s->nc[d] = nc[d]; s->per[d] = per[d]; }
    s->alat = alat;
    s->ncell = (long)nc[0] * nc[1] * nc[2];
    s->N = s->ncell * nb;
    s->mu = (double *)malloc(nb * sizeof(double));
    s->K = (double *)calloc(nb, sizeof(double));
    s->Kax = (double *)calloc(3 * nb, sizeof(double));
    for (int b = 0; b < nb; ++b) { s->mu[b] = 1.0; s->Kax[3*b+2] = 1.0; }
    s->n = (double *)calloc(3 * s->N, sizeof(double));
    for (long i = 0; i < s->N; ++i) s->n[3*i+2] = 1.0;
    s->dt = 1e-3; s->alpha = 0.1; s->jdir[0] = 1.0;
#ifdef _OPENMP
    s->nthreads = omp_get_max_threads();
#else
    s->nthreads = 1;
#endif
    return s;
}
void orc_destroy(orc_system *s) {
    if (!s) return;
    free(s->basis); free(s->mu); free(s->K); free(s->Kax); free(s->ab); free(s->aK); free(s->aax);
    free(s->pi); free(s->pj); free(s->pt); free(s->pJ); free(s->pD);
    free(s->qb); free(s->qt); free(s->qK); free(s->Khat); free(s->n); free(s->pinned); free(s->mu_site); free(s->vp_v); free(s->vp_F);
    free(s);
}
long orc_nspins(const orc_system *s) { return s->N; }
int orc_threads(const orc_system *s) { return s->nthreads; }
void orc_set_threads(orc_system *s, int n) {
#ifdef _OPENMP
    if (n < 1) n = 1;
    s->nthreads = n;
#else
    (void)n; s->nthreads = 1;
#endif
}
void orc_set_mu_s(orc_system *s, const double *mu) { memcpy(s->mu, mu, s->nb * sizeof(double)); free(s->Khat); s->Khat = NULL; }
/* per-site moments (":79 atoms of different types"), N values in boundary order; NULL goes back to the basis atoms' moments */
void orc_set_site_mu_s(orc_system *s, const double *mu_site) {
    free(s->mu_site); s->mu_site = NULL;
    if (mu_site) { s->mu_site = (double *)malloc(s->N * sizeof(double)); memcpy(s->mu_site, mu_site, s->N * sizeof(double)); }
}
void orc_set_field(orc_system *s, double B, const double dir[3]) {
    double nrm = sqrt(dot3(dir, dir));
    for (int k = 0; k < 3; ++k) s->Bext[k] = (nrm > 0) ? B * dir[k] / nrm : 0.0;
}
void orc_set_anisotropy(orc_system *s, int n, const int *bidx, const double *K, const double *axis) {
    free(s->ab); free(s->aK); free(s->aax);
    s->nani = n;
    s->ab = (int *)malloc((n + 1) * sizeof(int)); s->aK = (double *)malloc((n + 1) * sizeof(double)); s->aax = (double *)malloc(3 * (n + 1) * sizeof(double));
    for (int e = 0; e < n; ++e) {
        double nrm = sqrt(dot3(axis + 3*e, axis + 3*e));
        s->ab[e] = bidx[e]; s->aK[e] = K[e];
        for (int k = 0; k < 3; ++k) s->aax[3*e+k] = axis[3*e+k] / nrm;
    }
}
void orc_set_pairs(orc_system *s, int np, const int *pi, const int *pj, const int *pt,
                   const double *J, const double *D) {
    free(s->pi); free(s->pj); free(s->pt); free(s->pJ); free(s->pD);
    s->npairs = np;
    s->pi = (int *)malloc((np + 1) * sizeof(int));     memcpy(s->pi, pi, np * sizeof(int));
    s->pj = (int *)malloc((np + 1) * sizeof(int));     memcpy(s->pj, pj, np * sizeof(int));
    s->pt = (int *)malloc((3 * np + 1) * sizeof(int)); memcpy(s->pt, pt, 3 * np * sizeof(int));
    s->pJ = (double *)malloc((np + 1) * sizeof(double)); memcpy(s->pJ, J, np * sizeof(double));
    s->pD = (double *)calloc(3 * np + 1, sizeof(double));
    if (D) memcpy(s->pD, D, 3 * np * sizeof(double));
}
void orc_set_quadruplets(orc_system *s, int nq, const int *qb, const int *qt, const double *K) {
    free(s->qb); free(s->qt); free(s->qK);
    s->nquads = nq;
    s->qb = (int *)malloc((4 * nq + 1) * sizeof(int)); memcpy(s->qb, qb, 4 * nq * sizeof(int));
    s->qt = (int *)malloc((9 * nq + 1) * sizeof(int)); memcpy(s->qt, qt, 9 * nq * sizeof(int));
    s->qK = (double *)malloc((nq + 1) * sizeof(double)); memcpy(s->qK, K, nq * sizeof(double));
}
void orc_set_ddi(orc_system *s, int enabled, const int nimg[3], int direct) {
    s->ddi = enabled; s->ddi_direct = direct;
    for (int d = 0; d < 3; ++d) s->nimg[d] = nimg[d];
    free(s->Khat); s->Khat = NULL;
}
void orc_set_spins(orc_system *s, const double *n) { memcpy(s->n, n, 3 * s->N * sizeof(double)); }
void orc_get_spins(const orc_system *s, double *n) { memcpy(n, s->n, 3 * s->N * sizeof(double)); }
void orc_llg_configure(orc_system *s, double dt_fs, double alpha, double T, uint64_t seed,
                       double u, const double jdir[3], double beta) {
    s->dt = dt_fs * 1e-3; s->alpha = alpha; s->T = T; s->seed = seed; s->u = u; s->beta = beta;
    double nrm = sqrt(dot3(jdir, jdir));
    for (int k = 0; k < 3; ++k) s->jdir[k] = (nrm > 0) ? jdir[k] / nrm : 0.0;
    s->step = 0;
}
void orc_set_solver(orc_system *s, int solver) { s->solver = solver; }
void orc_set_image(orc_system *s, uint32_t image) { s->image = image; }
void orc_set_damping_only(orc_system *s, int on) { s->damping_only = on ? 1 : 0; }
void orc_set_pinned(orc_system *s, const unsigned char *mask) {
    free(s->pinned); s->pinned = NULL;
    if (!mask) return;
    s->pinned = (unsigned char *)malloc((size_t)s->N);
    memcpy(s->pinned, mask, (size_t)s->N);
}
uint64_t orc_get_step(const orc_system *s) { return s->step; }
void orc_set_step(orc_system *s, uint64_t st) { s->step = st; }

/* ------------------------------------------------------------------ energy, Eq. 1 and Eq. 2
 * Written as the sums are printed: one loop per term over cells and list entries.
 * Reading R3: anisotropy axis/strength per basis atom.  Reading R4: each pair once, weight J.
 * Reading R1: dipolar term in its textbook form
 *     -1/2 C_dd sum_{i != j} mu_i mu_j [3 (n_i.r^)(n_j.r^) - n_i.n_j] / r^3 .             */
void orc_ddi_direct(const orc_system *s, const double *n, double *F);
void orc_ddi_fft(orc_system *s, const double *n, double *F);

void orc_energy(orc_system *s, const double *n, double E[6]) {
    long double ez = 0, ea = 0, ex = 0, ed = 0, eq = 0, edd = 0;
    int c[3], cj[3], ck[3], cl[3];
    for (long cell = 0; cell < s->ncell; ++cell) {
        cell_coords(s, cell, c);
        for (int b = 0; b < s->nb; ++b) {
            const double *ni = n + 3 * spin_index(s, c, b);
            ez -= (long double)(mu_at(s, spin_index(s, c, b)) * ORC_MU_B * dot3(s->Bext, ni));
            for (int e = 0; e < s->nani; ++e) if (s->ab[e] == b) {
                double p = dot3(s->aax + 3*e, ni);
                ea -= (long double)(s->aK[e] * p * p);
            }
        }
        for (int p = 0; p < s->npairs; ++p) {
            if (!shifted_cell(s, c, s->pt + 3*p, +1, cj)) continue;
            const double *ni = n + 3 * spin_index(s, c, s->pi[p]);
            const double *nj = n + 3 * spin_index(s, cj, s->pj[p]);
            double cr[3]; cross3(ni, nj, cr);
            ex -= (long double)(s->pJ[p] * dot3(ni, nj));
            ed -= (long double)(dot3(s->pD + 3*p, cr));
        }
        for (int q = 0; q < s->nquads; ++q) {
            if (!shifted_cell(s, c, s->qt + 9*q + 0, +1, cj)) continue;
            if (!shifted_cell(s, c, s->qt + 9*q + 3, +1, ck)) continue;
            if (!shifted_cell(s, c, s->qt + 9*q + 6, +1, cl)) continue;
            const double *ni = n + 3 * spin_index(s, c,  s->qb[4*q+0]);
            const double *nj = n + 3 * spin_index(s, cj, s->qb[4*q+1]);
            const double *nk = n + 3 * spin_index(s, ck, s->qb[4*q+2]);
            const double *nl = n + 3 * spin_index(s, cl, s->qb[4*q+3]);
            eq -= (long double)(s->qK[q] * dot3(ni, nj) * dot3(nk, nl));
        }
    }
    if (s->ddi) {
        /* E_dd = -1/2 sum_i n_i . F_i^dd  (F^dd is linear in n; the 1/2 is the one printed in Eq. 1) */
        double *F = (double *)calloc(3 * s->N, sizeof(double));
        if (s->ddi_direct) orc_ddi_direct(s, n, F); else orc_ddi_fft(s, n, F);
        for (long i = 0; i < s->N; ++i) edd -= 0.5L * (long double)dot3(n + 3*i, F + 3*i);
        free(F);
    }
    E[0] = (double)ez; E[1] = (double)ea; E[2] = (double)ex; E[3] = (double)ed; E[4] = (double)eq; E[5] = (double)edd;
}

/* Dipolar energy straight from the double sum of Eq. 1 (reading R1), pair by pair. Tiny lattices only. */
double orc_energy_ddi_pairsum(const orc_system *s, const double *n) {
    long double e = 0;
    int ci[3], cj[3];
    for (long celli = 0; celli < s->ncell; ++celli) for (int a = 0; a < s->nb; ++a) {
        cell_coords(s, celli, ci);
        const double *ni = n + 3 * spin_index(s, ci, a);
        for (long cellj = 0; cellj < s->ncell; ++cellj) for (int b = 0; b < s->nb; ++b) {
            cell_coords(s, cellj, cj);
            const double *nj = n + 3 * spin_index(s, cj, b);
            for (int t0 = -(s->per[0] ? s->nimg[0] : 0); t0 <= (s->per[0] ? s->nimg[0] : 0); ++t0)
            for (int t1 = -(s->per[1] ? s->nimg[1] : 0); t1 <= (s->per[1] ? s->nimg[1] : 0); ++t1)
            for (int t2 = -(s->per[2] ? s->nimg[2] : 0); t2 <= (s->per[2] ? s->nimg[2] : 0); ++t2) {
                if (celli == cellj && a == b && t0 == 0 && t1 == 0 && t2 == 0) continue;
                double f[3] = { cj[0] - ci[0] + (double)t0 * s->nc[0] + s->basis[3*b+0] - s->basis[3*a+0],
                                cj[1] - ci[1] + (double)t1 * s->nc[1] + s->basis[3*b+1] - s->basis[3*a+1],
                                cj[2] - ci[2] + (double)t2 * s->nc[2] + s->basis[3*b+2] - s->basis[3*a+2] };
                double r[3]; frac_to_cart(s, f, r);
                double r2 = dot3(r, r), rn = sqrt(r2);
                double rh[3] = { r[0]/rn, r[1]/rn, r[2]/rn };
                e -= 0.5L * (long double)(ORC_C_DD * mu_at(s, spin_index(s, ci, a)) * mu_at(s, spin_index(s, cj, b)) *
                        (3.0 * dot3(ni, rh) * dot3(nj, rh) - dot3(ni, nj)) / (r2 * rn));
            }
        }
    }
    return (double)e;
}

/* ------------------------------------------------------------------ gradient, scatter form
 * F_i = -dH/dn_i in the embedding space, term by term as the derivative of orc_energy's sums:
 *   pair (i,j,J,D):   F_i += J n_j + n_j x D ;  F_j += J n_i - n_i x D
 *                     (from D.(n_i x n_j) = n_i.(n_j x D) = -n_j.(n_i x D))
 *   quad (i,j,k,l,K): F_i += K (n_k.n_l) n_j ; F_j += K (n_k.n_l) n_i ;
 *                     F_k += K (n_i.n_j) n_l ; F_l += K (n_i.n_j) n_k
 * Serial; used to pin the parallel gather form below.                                   */
void orc_gradient_scatter(orc_system *s, const double *n, double *F, int mask) {
    memset(F, 0, 3 * s->N * sizeof(double));
    int c[3], cj[3], ck[3], cl[3];
    for (long cell = 0; cell < s->ncell; ++cell) {
        cell_coords(s, cell, c);
        for (int b = 0; b < s->nb; ++b) {
            long i = spin_index(s, c, b);
            if (mask & T_ZEE) for (int k = 0; k < 3; ++k) F[3*i+k] += mu_at(s, i) * ORC_MU_B * s->Bext[k];
            if (mask & T_ANI) for (int e = 0; e < s->nani; ++e) if (s->ab[e] == b) {
                double p = dot3(s->aax + 3*e, n + 3*i);
                for (int k = 0; k < 3; ++k) F[3*i+k] += 2.0 * s->aK[e] * p * s->aax[3*e+k];
            }
        }
        for (int p = 0; p < s->npairs; ++p) {
            if (!shifted_cell(s, c, s->pt + 3*p, +1, cj)) continue;
            long i = spin_index(s, c, s->pi[p]), j = spin_index(s, cj, s->pj[p]);
            const double *D = s->pD + 3*p;
            if (mask & T_EXC) for (int k = 0; k < 3; ++k) {
                F[3*i+k] += s->pJ[p] * n[3*j+k];
                F[3*j+k] += s->pJ[p] * n[3*i+k];
            }
            if (mask & T_DMI) {
                double a[3], bb[3];
                cross3(n + 3*j, D, a); cross3(n + 3*i, D, bb);
                for (int k = 0; k < 3; ++k) { F[3*i+k] += a[k]; F[3*j+k] -= bb[k]; }
            }
        }
        if (mask & T_QUAD) for (int q = 0; q < s->nquads; ++q) {
            if (!shifted_cell(s, c, s->qt + 9*q + 0, +1, cj)) continue;
            if (!shifted_cell(s, c, s->qt + 9*q + 3, +1, ck)) continue;
            if (!shifted_cell(s, c, s->qt + 9*q + 6, +1, cl)) continue;
            long i = spin_index(s, c,  s->qb[4*q+0]), j = spin_index(s, cj, s->qb[4*q+1]);
            long k = spin_index(s, ck, s->qb[4*q+2]), l = spin_index(s, cl, s->qb[4*q+3]);
            double dij = dot3(n + 3*i, n + 3*j), dkl = dot3(n + 3*k, n + 3*l), K = s->qK[q];
            for (int x = 0; x < 3; ++x) {
                double fi = K * dkl * n[3*j+x], fj = K * dkl * n[3*i+x];
                double fk = K * dij * n[3*l+x], fl = K * dij * n[3*k+x];
                F[3*i+x] += fi; F[3*j+x] += fj; F[3*k+x] += fk; F[3*l+x] += fl;
            }
        }
    }
    if ((mask & T_DDI) && s->ddi) {
        double *Fd = (double *)calloc(3 * s->N, sizeof(double));
        if (s->ddi_direct) orc_ddi_direct(s, n, Fd); else orc_ddi_fft(s, n, Fd);
        for (long i = 0; i < 3 * s->N; ++i) F[i] += Fd[i];
        free(Fd);
    }
}

/* ------------------------------------------------------------------ gradient, gather form
 * Same sums, regrouped per spin so that spins can be processed independently (OpenMP):
 * a spin on basis atom b collects, for every list entry in which b appears, the partner's
 * contribution.  For a pair (bi, bj, t): as "i" the partner is (cell + t, bj) with +D; as "j"
 * the partner is (cell - t, bi) with -D.  A quadruplet anchored at cell c0 has its four
 * members at c0, c0+tj, c0+tk, c0+tl; a spin in role r sits at c0 + t_r, so c0 = cell - t_r.
 * A quadruplet with any member off an open edge does not exist (reading R20).             */
static void gather_one(const orc_system *s, const double *n, long cell, int b, int mask, double F[3]) {
    int c[3], c2[3], c0[3], cm[4][3];
    static const int zero3[3] = {0, 0, 0};
    cell_coords(s, cell, c);
    const double *ni = n + 3 * spin_index(s, c, b);
    F[0] = F[1] = F[2] = 0.0;
    if (mask & T_ZEE) for (int k = 0; k < 3; ++k) F[k] += mu_at(s, spin_index(s, c, b)) * ORC_MU_B * s->Bext[k];
    if (mask & T_ANI) for (int e = 0; e < s->nani; ++e) if (s->ab[e] == b) {
        double p = dot3(s->aax + 3*e, ni);
        for (int k = 0; k < 3; ++k) F[k] += 2.0 * s->aK[e] * p * s->aax[3*e+k];
    }
    if (mask & (T_EXC | T_DMI)) for (int p = 0; p < s->npairs; ++p) {
        const double *D = s->pD + 3*p;
        if (s->pi[p] == b && shifted_cell(s, c, s->pt + 3*p, +1, c2)) {
            const double *nj = n + 3 * spin_index(s, c2, s->pj[p]);
            if (mask & T_EXC) for (int k = 0; k < 3; ++k) F[k] += s->pJ[p] * nj[k];
            if (mask & T_DMI) { double x[3]; cross3(nj, D, x); for (int k = 0; k < 3; ++k) F[k] += x[k]; }
        }
        if (s->pj[p] == b && shifted_cell(s, c, s->pt + 3*p, -1, c2)) {
            const double *nj = n + 3 * spin_index(s, c2, s->pi[p]);
            if (mask & T_EXC) for (int k = 0; k < 3; ++k) F[k] += s->pJ[p] * nj[k];
            if (mask & T_DMI) { double x[3]; cross3(nj, D, x); for (int k = 0; k < 3; ++k) F[k] -= x[k]; }
        }
    }
    if (mask & T_QUAD) for (int q = 0; q < s->nquads; ++q) {
        for (int role = 0; role < 4; ++role) {
            if (s->qb[4*q + role] != b) continue;
            const int *tr = (role == 0) ? zero3 : s->qt + 9*q + 3*(role-1);
            if (!shifted_cell(s, c, tr, -1, c0)) continue;
            int ok = 1;
            for (int m = 0; m < 4 && ok; ++m) {
                const int *tm = (m == 0) ? zero3 : s->qt + 9*q + 3*(m-1);
                ok = shifted_cell(s, c0, tm, +1, cm[m]);
            }
            if (!ok) continue;
            /* the member that must come back to this very site (guards against open-edge aliasing) */
            if (cm[role][0] != c[0] || cm[role][1] != c[1] || cm[role][2] != c[2]) continue;
            const double *m0 = n + 3 * spin_index(s, cm[0], s->qb[4*q+0]);
            const double *m1 = n + 3 * spin_index(s, cm[1], s->qb[4*q+1]);
            const double *m2 = n + 3 * spin_index(s, cm[2], s->qb[4*q+2]);
            const double *m3 = n + 3 * spin_index(s, cm[3], s->qb[4*q+3]);
            double K = s->qK[q];
            const double *partner; double w;
            if (role == 0)      { partner = m1; w = dot3(m2, m3); }
            else if (role == 1) { partner = m0; w = dot3(m2, m3); }
            else if (role == 2) { partner = m3; w = dot3(m0, m1); }
            else                { partner = m2; w = dot3(m0, m1); }
            for (int k = 0; k < 3; ++k) F[k] += K * w * partner[k];
        }
    }
}

void orc_gradient(orc_system *s, const double *n, double *F, int mask) {
    long N = s->N; int nb = s->nb; (void)nb;
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
    for (long i = 0; i < N; ++i) gather_one(s, n, i / nb, (int)(i % nb), mask, F + 3*i);
    if ((mask & T_DDI) && s->ddi) {
        double *Fd = (double *)calloc(3 * N, sizeof(double));
        if (s->ddi_direct) orc_ddi_direct(s, n, Fd); else orc_ddi_fft(s, n, Fd);
        for (long i = 0; i < 3 * N; ++i) F[i] += Fd[i];
        free(Fd);
    }
}

/* ------------------------------------------------------------------ dipole-dipole, direct sum (:81, :89)
 * F_i = mu_i C_dd sum_{j, images; r != 0} mu_j [3 r^ (n_j.r^) - n_j] / r^3 ,  r = r_j + image - r_i.
 * Images: t_d in [-nimg_d, nimg_d] in periodic directions, 0 in open ones (reading R16);
 * self images (i == j, t != 0) are included.                                              */
void orc_ddi_direct(const orc_system *s, const double *n, double *F) {
    long N = s->N; int nb = s->nb; (void)nb;
    int lim[3]; for (int d = 0; d < 3; ++d) lim[d] = s->per[d] ? s->nimg[d] : 0;
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
    for (long i = 0; i < N; ++i) {
        int ci[3], cj[3]; cell_coords(s, i / nb, ci); int a = (int)(i % nb);
        double acc[3] = {0, 0, 0};
        for (long j = 0; j < N; ++j) {
            cell_coords(s, j / nb, cj); int b = (int)(j % nb);
            const double *nj = n + 3*j;
            for (int t0 = -lim[0]; t0 <= lim[0]; ++t0)
            for (int t1 = -lim[1]; t1 <= lim[1]; ++t1)
            for (int t2 = -lim[2]; t2 <= lim[2]; ++t2) {
                if (i == j && t0 == 0 && t1 == 0 && t2 == 0) continue;
                double f[3] = { cj[0] - ci[0] + (double)t0 * s->nc[0] + s->basis[3*b+0] - s->basis[3*a+0],
                                cj[1] - ci[1] + (double)t1 * s->nc[1] + s->basis[3*b+1] - s->basis[3*a+1],
                                cj[2] - ci[2] + (double)t2 * s->nc[2] + s->basis[3*b+2] - s->basis[3*a+2] };
                double r[3]; frac_to_cart(s, f, r);
                double r2 = dot3(r, r), rn = sqrt(r2);
                double rh[3] = { r[0]/rn, r[1]/rn, r[2]/rn };
                double p = dot3(nj, rh), w = mu_at(s, j) / (r2 * rn);
                for (int k = 0; k < 3; ++k) acc[k] += w * (3.0 * rh[k] * p - nj[k]);
            }
        }
        for (int k = 0; k < 3; ++k) F[3*i+k] = mu_at(s, i) * ORC_C_DD * acc[k];
    }
}

/* ------------------------------------------------------------------ own FFT (paper uses FFTW3, :87)
 * In-place complex transform of length n, sign = -1 forward / +1 backward, unnormalised.
 * Power-of-two lengths: textbook iterative radix-2 (bit reversal + butterflies, twiddles
 * from cos/sin of the exact angle).  Any other length: the DFT sum written out.           */
static void fft_line(double *re, double *im, int n, int sign) {
    if (n <= 1) return;
    if ((n & (n - 1)) == 0) {
        for (int i = 1, j = 0; i < n; ++i) {
            int bit = n >> 1;
            for (; j & bit; bit >>= 1) j ^= bit;
            j ^= bit;
            if (i < j) { double t = re[i]; re[i] = re[j]; re[j] = t; t = im[i]; im[i] = im[j]; im[j] = t; }
        }
        for (int len = 2; len <= n; len <<= 1) {
            int half = len >> 1;
            for (int k = 0; k < half; ++k) {
                double ang = sign * 2.0 * ORC_PI * (double)k / (double)len;
                double wr = cos(ang), wi = sin(ang);
                for (int i = k; i < n; i += len) {
                    int j = i + half;
                    double xr = re[j]*wr - im[j]*wi, xi = re[j]*wi + im[j]*wr;
                    re[j] = re[i] - xr; im[j] = im[i] - xi;
                    re[i] += xr; im[i] += xi;
                }
            }
        }
    } else {
        double *or_ = (double *)malloc(2 * n * sizeof(double)), *oi = or_ + n;
        for (int k = 0; k < n; ++k) {
            double sr = 0, si = 0;
            for (int j = 0; j < n; ++j) {
                double ang = sign * 2.0 * ORC_PI * (double)(((long)k * j) % n) / (double)n;
                double wr = cos(ang), wi = sin(ang);
                sr += re[j]*wr - im[j]*wi; si += re[j]*wi + im[j]*wr;
            }
            or_[k] = sr; oi[k] = si;
        }
        memcpy(re, or_, n * sizeof(double)); memcpy(im, oi, n * sizeof(double));
        free(or_);
    }
}
/* 3-D transform of interleaved complex data z[2*(x + P0*(y + P1*zc))], one axis after the other */
static void fft3d(double *z, const int P[3], int sign, int nthreads) {
    long stride[3] = { 1, P[0], (long)P[0] * P[1] };
    long Ptot = (long)P[0] * P[1] * P[2];
    (void)nthreads;
    for (int ax = 0; ax < 3; ++ax) {
        int n = P[ax];
        if (n == 1) continue;
        long nlines = Ptot / n;
#pragma omp parallel num_threads(nthreads)
        {
            double *re = (double *)malloc(2 * n * sizeof(double)), *im = re + n;
#pragma omp for schedule(static)
            for (long line = 0; line < nlines; ++line) {
                /* base index of this line: enumerate the other two axes */
                int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
                long i1 = line % P[a1], i2 = line / P[a1];
                long base = i1 * stride[a1] + i2 * stride[a2];
                for (int k = 0; k < n; ++k) { re[k] = z[2*(base + k*stride[ax])]; im[k] = z[2*(base + k*stride[ax]) + 1]; }
                fft_line(re, im, n, sign);
                for (int k = 0; k < n; ++k) { z[2*(base + k*stride[ax])] = re[k]; z[2*(base + k*stride[ax]) + 1] = im[k]; }
            }
            free(re);
        }
    }
}
/* exported for the FFT pins */
void orc_fft3d(double *z, const int P[3], int sign) { fft3d(z, P, sign, 1); }

/* ------------------------------------------------------------------ dipole-dipole by padded FFT (:81-87)
 * One padded array per sublattice, one convolution per sublattice pair (:87).
 *   P_d = 2 N_d if N_d > 1 else 1 (reading R17).
 *   K_ab(Delta) = sum_images T(r), r = alat * ((Delta + t*N) + p_a - p_b) . bravais,
 *   T(r) = (3 r^ r^T - 1)/r^3, stored at index Delta mod P_d for Delta in (-N_d, N_d);
 *   Delta = (target cell) - (source cell).  T is even in r, so this equals T(r_j - r_i).
 *   F_a(c) = mu_a C_dd sum_b sum_c' K_ab(c - c') mu_b n_b(c')
 *          = mu_a C_dd IFFT[ sum_b K^_ab . FFT[mu_b n_b zero-padded] ](c).
 * Six independent components xx, xy, xz, yy, yz, zz.                                       */
static const int SYM_A[6] = {0, 0, 0, 1, 1, 2}, SYM_B[6] = {0, 1, 2, 1, 2, 2};

static void ddi_prepare(orc_system *s) {
    if (s->Khat) return;
    for (int d = 0; d < 3; ++d) s->P[d] = (s->nc[d] > 1) ? 2 * s->nc[d] : 1;
    s->Ptot = (long)s->P[0] * s->P[1] * s->P[2];
    long Pt = s->Ptot; int nb = s->nb;
    s->Khat = (double *)calloc((size_t)nb * nb * 6 * Pt * 2, sizeof(double));
    int lim[3]; for (int d = 0; d < 3; ++d) lim[d] = s->per[d] ? s->nimg[d] : 0;
    for (int a = 0; a < nb; ++a) for (int b = 0; b < nb; ++b) {
        double *Kab = s->Khat + ((size_t)(a * nb + b) * 6) * Pt * 2;
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
        for (long idx = 0; idx < Pt; ++idx) {
            int g[3] = { (int)(idx % s->P[0]), (int)((idx / s->P[0]) % s->P[1]), (int)(idx / ((long)s->P[0] * s->P[1])) };
            int Delta[3], skip = 0;
            for (int d = 0; d < 3; ++d) {
                if (s->P[d] == 1) { Delta[d] = 0; continue; }
                if (g[d] == s->nc[d]) { skip = 1; break; }          /* index N_d stays zero */
                Delta[d] = (g[d] < s->nc[d]) ? g[d] : g[d] - s->P[d];
            }
            if (skip) continue;
            double acc[6] = {0, 0, 0, 0, 0, 0};
            for (int t0 = -lim[0]; t0 <= lim[0]; ++t0)
            for (int t1 = -lim[1]; t1 <= lim[1]; ++t1)
            for (int t2 = -lim[2]; t2 <= lim[2]; ++t2) {
                double f[3] = { Delta[0] + (double)t0 * s->nc[0] + s->basis[3*a+0] - s->basis[3*b+0],
                                Delta[1] + (double)t1 * s->nc[1] + s->basis[3*a+1] - s->basis[3*b+1],
                                Delta[2] + (double)t2 * s->nc[2] + s->basis[3*a+2] - s->basis[3*b+2] };
                double r[3]; frac_to_cart(s, f, r);
                double r2 = dot3(r, r);
                if (r2 < 1e-20) continue;                             /* r = 0: the i == j term */
                double rn = sqrt(r2), r3 = r2 * rn;
                double rh[3] = { r[0]/rn, r[1]/rn, r[2]/rn };
                for (int m = 0; m < 6; ++m)
                    acc[m] += (3.0 * rh[SYM_A[m]] * rh[SYM_B[m]] - (SYM_A[m] == SYM_B[m] ? 1.0 : 0.0)) / r3;
            }
            for (int m = 0; m < 6; ++m) Kab[2 * ((size_t)m * Pt + idx)] = acc[m];
        }
        for (int m = 0; m < 6; ++m) fft3d(Kab + 2 * (size_t)m * Pt, s->P, -1, s->nthreads);
    }
}

void orc_ddi_fft(orc_system *s, const double *n, double *F) {
    ddi_prepare(s);
    long Pt = s->Ptot; int nb = s->nb;
    double *M = (double *)calloc((size_t)nb * 3 * Pt * 2, sizeof(double));
    double *H = (double *)malloc((size_t)3 * Pt * 2 * sizeof(double));
    int c[3];
    for (long cell = 0; cell < s->ncell; ++cell) {
        cell_coords(s, cell, c);
        long pidx = c[0] + (long)s->P[0] * (c[1] + (long)s->P[1] * c[2]);
        for (int b = 0; b < nb; ++b) for (int k = 0; k < 3; ++k)
            M[2 * ((size_t)(b * 3 + k) * Pt + pidx)] = mu_at(s, spin_index(s, c, b)) * n[3 * spin_index(s, c, b) + k];
    }
    for (int b = 0; b < nb; ++b) for (int k = 0; k < 3; ++k) fft3d(M + 2 * (size_t)(b * 3 + k) * Pt, s->P, -1, s->nthreads);
    for (int a = 0; a < nb; ++a) {
        memset(H, 0, (size_t)3 * Pt * 2 * sizeof(double));
        for (int b = 0; b < nb; ++b) {
            const double *Kab = s->Khat + ((size_t)(a * nb + b) * 6) * Pt * 2;
            const double *Mb = M + 2 * (size_t)(b * 3) * Pt;
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
            for (long q = 0; q < Pt; ++q) {
                /* full symmetric 3x3 from the six stored components */
                static const int comp[3][3] = { {0, 1, 2}, {1, 3, 4}, {2, 4, 5} };
                for (int al = 0; al < 3; ++al) {
                    double hr = 0, hi = 0;
                    for (int be = 0; be < 3; ++be) {
                        double kr = Kab[2 * ((size_t)comp[al][be] * Pt + q)], ki = Kab[2 * ((size_t)comp[al][be] * Pt + q) + 1];
                        double mr = Mb[2 * ((size_t)be * Pt + q)], mi = Mb[2 * ((size_t)be * Pt + q) + 1];
                        hr += kr * mr - ki * mi; hi += kr * mi + ki * mr;
                    }
                    H[2 * ((size_t)al * Pt + q)] += hr; H[2 * ((size_t)al * Pt + q) + 1] += hi;
                }
            }
        }
        for (int k = 0; k < 3; ++k) fft3d(H + 2 * (size_t)k * Pt, s->P, +1, s->nthreads);
        for (long cell = 0; cell < s->ncell; ++cell) {
            cell_coords(s, cell, c);
            long pidx = c[0] + (long)s->P[0] * (c[1] + (long)s->P[1] * c[2]);
            for (int k = 0; k < 3; ++k)
                F[3 * spin_index(s, c, a) + k] = mu_at(s, spin_index(s, c, a)) * ORC_C_DD * H[2 * ((size_t)k * Pt + pidx)] / (double)Pt;
        }
    }
    free(M); free(H);
}

/* ------------------------------------------------------------------ Philox4x32-10 (reading R13)
 * Salmon et al. counter-based generator: 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0)),
 * key bumped by (W0, W1) between rounds.                                                  */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* uniform in (0,1) from 64 bits: top 53 bits plus one half, times 2^-53 */
static inline double u01(uint32_t hi, uint32_t lo) {
    uint64_t v = (((uint64_t)hi << 32) | lo) >> 11;
    return ((double)v + 0.5) * (1.0 / 9007199254740992.0);
}
/* three standard normals for (seed, step, spin): key = seed, counter = (spin, block, step_lo, step_hi);
 * Box-Muller; block 0 -> (xi_x, xi_y), block 1 -> xi_z.                                      */
/* Independent images (chain of images :197, temperature sweeps :143, Fig. 13) draw independent noise from the same seed: image m
 * uses the counter words block + 2 m (reading R30); image 0 is the single-system stream.                                    */
void orc_thermal_xi_image(uint64_t seed, uint64_t step, uint32_t spin, uint32_t image, double xi[3]) {
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, x[4];
    uint32_t c0[4] = { spin, 2u * image, (uint32_t)step, (uint32_t)(step >> 32) };
    orc_philox4x32_10(c0, key, x);
    double u1 = u01(x[0], x[1]), u2 = u01(x[2], x[3]);
    double rad = sqrt(-2.0 * log(u1));
    xi[0] = rad * cos(2.0 * ORC_PI * u2);
    xi[1] = rad * sin(2.0 * ORC_PI * u2);
    uint32_t c1[4] = { spin, 2u * image + 1u, (uint32_t)step, (uint32_t)(step >> 32) };
    orc_philox4x32_10(c1, key, x);
    u1 = u01(x[0], x[1]); u2 = u01(x[2], x[3]);
    xi[2] = sqrt(-2.0 * log(u1)) * cos(2.0 * ORC_PI * u2);
}
void orc_thermal_xi(uint64_t seed, uint64_t step, uint32_t spin, double xi[3]) { orc_thermal_xi_image(seed, step, spin, 0u, xi); }
/* Eq. 11 with the 1/sqrt(dt) of :160 (reading R10): sigma = sqrt(2 alpha k_B T mu / (gamma dt)), meV */
double orc_thermal_sigma(const orc_system *s, int b) {
    return sqrt(2.0 * s->alpha * ORC_K_B * s->T * s->mu[b] * ORC_MU_B / (ORC_GAMMA * s->dt));
}
/* the same for spin i, with its own moment when per-site moments are set */
static double thermal_sigma_site(const orc_system *s, long i) {
    return sqrt(2.0 * s->alpha * ORC_K_B * s->T * mu_at(s, i) * ORC_MU_B / (ORC_GAMMA * s->dt));
}

/* ------------------------------------------------------------------ (j_e . grad) n on the lattice (reading R14)
 * j^ is expanded in the Bravais vectors of the directions with more than one cell
 * (least squares when there are fewer than three), j^ = sum_d c_d a_d (a_d in Angstrom), so that
 * (j^.grad) n = sum_d c_d dn/dx_d with x_d the cell coordinate; dn/dx_d by central differences
 * on the same sublattice, one-sided at an open edge.                                          */
static void stt_coeffs(const orc_system *s, double cd[3]) {
    int act[3], na = 0;
    for (int d = 0; d < 3; ++d) { cd[d] = 0.0; if (s->nc[d] > 1) act[na++] = d; }
    if (na == 0) return;
    double G[3][3], rhs[3];
    for (int p = 0; p < na; ++p) {
        double ap[3]; for (int k = 0; k < 3; ++k) ap[k] = s->alat * s->brav[3*act[p]+k];
        rhs[p] = dot3(ap, s->jdir);
        for (int q = 0; q < na; ++q) {
            double aq[3]; for (int k = 0; k < 3; ++k) aq[k] = s->alat * s->brav[3*act[q]+k];
            G[p][q] = dot3(ap, aq);
        }
    }
    /* solve the (na x na) normal equations G c = rhs by Gaussian elimination with pivoting */
    for (int p = 0; p < na; ++p) {
        int piv = p;
        for (int r = p + 1; r < na; ++r) if (fabs(G[r][p]) > fabs(G[piv][p])) piv = r;
        if (piv != p) { for (int q = 0; q < na; ++q) { double t = G[p][q]; G[p][q] = G[piv][q]; G[piv][q] = t; } double t = rhs[p]; rhs[p] = rhs[piv]; rhs[piv] = t; }
        for (int r = p + 1; r < na; ++r) {
            double f = G[r][p] / G[p][p];
            for (int q = p; q < na; ++q) G[r][q] -= f * G[p][q];
            rhs[r] -= f * rhs[p];
        }
    }
    double sol[3];
    for (int p = na - 1; p >= 0; --p) {
        double v = rhs[p];
        for (int q = p + 1; q < na; ++q) v -= G[p][q] * sol[q];
        sol[p] = v / G[p][p];
    }
    for (int p = 0; p < na; ++p) cd[act[p]] = sol[p];
}
void orc_stt_gradient(orc_system *s, const double *n, double *sg) {
    double cd[3]; stt_coeffs(s, cd);
    long N = s->N; int nb = s->nb; (void)nb;
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
    for (long i = 0; i < N; ++i) {
        int c[3], cp[3], cm[3]; cell_coords(s, i / nb, c); int b = (int)(i % nb);
        double acc[3] = {0, 0, 0};
        for (int d = 0; d < 3; ++d) {
            if (s->nc[d] <= 1 || cd[d] == 0.0) continue;
            int e[3] = {0, 0, 0}; e[d] = 1;
            int hp = shifted_cell(s, c, e, +1, cp), hm = shifted_cell(s, c, e, -1, cm);
            const double *n0 = n + 3*i;
            const double *np_ = hp ? n + 3 * spin_index(s, cp, b) : n0;
            const double *nm_ = hm ? n + 3 * spin_index(s, cm, b) : n0;
            double w = (hp && hm) ? 0.5 : ((hp || hm) ? 1.0 : 0.0);
            for (int k = 0; k < 3; ++k) acc[k] += cd[d] * w * (np_[k] - nm_[k]);
        }
        for (int k = 0; k < 3; ++k) sg[3*i+k] = acc[k];
    }
}

/* ------------------------------------------------------------------ Eq. 10 as dn/dt = n x A (B1)
 * A = -gamma/((1+alpha^2) mu) [F + alpha n x F] + u/(1+alpha^2) [-(alpha-beta) s + (1+alpha beta) n x s]
 * with F in meV (incl. thermal), mu = mu_s mu_B in meV/T, s = (j^.grad) n in 1/Angstrom, u in A/ps. */
static inline void rot_field(const orc_system *s, long i, const double *n, const double *F, const double *sg, double *A) {
    double nxF[3], nxs[3] = {0, 0, 0};
    cross3(n, F, nxF);
    double pre = -ORC_GAMMA / ((1.0 + s->alpha * s->alpha) * mu_at(s, i) * ORC_MU_B);
    double us = s->u / (1.0 + s->alpha * s->alpha);
    if (s->u != 0.0) cross3(n, sg, nxs);
    for (int k = 0; k < 3; ++k) {
        /* ":168 these methods can also be used for energy minimization by considering only the damping part of the LLG equation" */
        A[k] = pre * ((s->damping_only ? 0.0 : F[k]) + s->alpha * nxF[k]);
        if (s->u != 0.0) A[k] += us * (-(s->alpha - s->beta) * sg[k] + (1.0 + s->alpha * s->beta) * nxs[k]);
    }
}
/* R(A) n: exact flow of dn/dt = n x A = (-A) x n over dt, i.e. Rodrigues rotation about
 * e = -A/|A| by theta = |A| dt (reading R7).                                                 */
static inline void rotate(const double *A, double dt, const double *n, double *out) {
    double a = sqrt(dot3(A, A));
    if (a == 0.0) { out[0] = n[0]; out[1] = n[1]; out[2] = n[2]; return; }
    double e[3] = { -A[0]/a, -A[1]/a, -A[2]/a }, th = a * dt, c = cos(th), sn = sin(th);
    double exn[3]; cross3(e, n, exn);
    double en = dot3(e, n);
    for (int k = 0; k < 3; ++k) out[k] = n[k] * c + exn[k] * sn + e[k] * en * (1.0 - c);
}

/* full force incl. thermal term; Fth may be NULL */
static void total_force(orc_system *s, const double *n, const double *Fth, double *F) {
    orc_gradient(s, n, F, T_ALL);
    if (Fth) for (long i = 0; i < 3 * s->N; ++i) F[i] += Fth[i];
}

/* Semi-implicit midpoint update (App. C, C5-C10): solve M x = M^T n with M = I + skew(A'), A' = (dt/2) A,
 * by Cramer's rule exactly as the paper writes it: a = M^T n = n + n x A' (C8), x_alpha = det(M^alpha)/det(M) (C9),
 * M^alpha = M with column alpha replaced by a (C10).  The paper prints M with A; the factor dt/2 follows from C5
 * (n^p - (dt/2) n^p x A = n + (dt/2) n x A), reading R25 in DESIGN.md.                                                */
static double det3(const double m[3][3]) {
    return m[0][0] * (m[1][1] * m[2][2] - m[1][2] * m[2][1]) - m[0][1] * (m[1][0] * m[2][2] - m[1][2] * m[2][0])
         + m[0][2] * (m[1][0] * m[2][1] - m[1][1] * m[2][0]);
}
static inline void imp_update(const double *A, double dt, const double *n, double *out) {
    double Ah[3] = { 0.5 * dt * A[0], 0.5 * dt * A[1], 0.5 * dt * A[2] };
    double M[3][3] = { { 1.0, -Ah[2], Ah[1] }, { Ah[2], 1.0, -Ah[0] }, { -Ah[1], Ah[0], 1.0 } };      /* C7 */
    double nxA[3]; cross3(n, Ah, nxA);
    double a[3] = { n[0] + nxA[0], n[1] + nxA[1], n[2] + nxA[2] };                                   /* C8 */
    double d = det3(M);
    for (int al = 0; al < 3; ++al) {
        double Ma[3][3];
        for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) Ma[r][c] = (c == al) ? a[r] : M[r][c];   /* C10 */
        out[al] = det3(Ma) / d;                                                                       /* C9 */
    }
}

/* One step of the selected solver.  All three are two-stage predictor/corrector schemes on dn/dt = n x A (B1) that share
 * the thermal field of the step between the stages (reading R11):
 *   Depondt (App. B, B5-B7): n^p = R(A) n; A^p = A(n^p); n <- R((A+A^p)/2) n(t) (reading R8); renormalise (R19).
 *   Heun (B3-B4 with f = n x A): n^p = n + dt n x A; n <- n + dt/2 (n x A + n^p x A^p); renormalise every step.
 *   SIB (App. C, C5, C11): n^p from the implicit-midpoint structure with A(n); n <- the same structure with A evaluated at
 *        the midpoint configuration {(n_j + n_j^p)/2}; length is preserved by construction, no renormalisation.        */
static void orc_rk4_step(orc_system *s);
void orc_llg_step(orc_system *s) {
    if (s->solver == 3) { orc_rk4_step(s); return; }
    long N = s->N; int nb = s->nb; (void)nb;
    double *F = (double *)malloc(3 * N * sizeof(double)), *A = (double *)malloc(3 * N * sizeof(double));
    double *np_ = (double *)malloc(3 * N * sizeof(double)), *sg = (double *)calloc(3 * N, sizeof(double));
    double *Fth = NULL;
    if (s->T > 0.0) {
        Fth = (double *)malloc(3 * N * sizeof(double));
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
        for (long i = 0; i < N; ++i) {
            double xi[3]; orc_thermal_xi_image(s->seed, s->step, (uint32_t)i, s->image, xi);
            double sig = thermal_sigma_site(s, i);
            for (int k = 0; k < 3; ++k) Fth[3*i+k] = sig * xi[k];
        }
    }
    total_force(s, s->n, Fth, F);
    if (s->u != 0.0) orc_stt_gradient(s, s->n, sg);
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
    for (long i = 0; i < N; ++i) {
        rot_field(s, i, s->n + 3*i, F + 3*i, sg + 3*i, A + 3*i);
        if (s->pinned && s->pinned[i]) { for (int k = 0; k < 3; ++k) np_[3*i+k] = s->n[3*i+k]; continue; }   /* pinned: n^p = n */
        if (s->solver == 0) rotate(A + 3*i, s->dt, s->n + 3*i, np_ + 3*i);                       /* B5 */
        else if (s->solver == 1) {                                                               /* B3 */
            double f0[3]; cross3(s->n + 3*i, A + 3*i, f0);
            for (int k = 0; k < 3; ++k) np_[3*i+k] = s->n[3*i+k] + s->dt * f0[k];
        } else imp_update(A + 3*i, s->dt, s->n + 3*i, np_ + 3*i);                                /* C5 */
    }
    /* configuration the second field is evaluated at: n^p (B6), or the midpoint (n + n^p)/2 (C11) */
    double *second = np_;
    if (s->solver == 2) for (long i = 0; i < 3 * N; ++i) np_[i] = 0.5 * (s->n[i] + np_[i]);
    total_force(s, second, Fth, F);
    if (s->u != 0.0) orc_stt_gradient(s, second, sg);
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
    for (long i = 0; i < N; ++i) {
        double Ap[3], Ac[3], out[3];
        if (s->pinned && s->pinned[i]) continue;                               /* pinned: n_i(t+dt) = n_i(t) */
        rot_field(s, i, second + 3*i, F + 3*i, sg + 3*i, Ap);
        if (s->solver == 0) {
            for (int k = 0; k < 3; ++k) Ac[k] = 0.5 * (A[3*i+k] + Ap[k]);     /* B6 */
            rotate(Ac, s->dt, s->n + 3*i, out);                               /* B7 */
        } else if (s->solver == 1) {                                          /* B4 */
            double f0[3], f1[3]; cross3(s->n + 3*i, A + 3*i, f0); cross3(np_ + 3*i, Ap, f1);
            for (int k = 0; k < 3; ++k) out[k] = s->n[3*i+k] + 0.5 * s->dt * (f0[k] + f1[k]);
        } else {
            imp_update(Ap, s->dt, s->n + 3*i, out);                           /* C11 */
        }
        if (s->solver == 2) { for (int k = 0; k < 3; ++k) s->n[3*i+k] = out[k]; continue; }
        double nrm = sqrt(dot3(out, out));
        for (int k = 0; k < 3; ++k) s->n[3*i+k] = out[k] / nrm;
    }
    s->step += 1;
    free(F); free(A); free(np_); free(sg); free(Fth);
}
/* Classical 4th-order Runge-Kutta on dn/dt = f(n) = n x A(n) (B1), "a 4th order Runge-Kutta solver" (:168; no formulas in the
 * paper, so the textbook tableau): k1 = f(n), k2 = f(n + dt/2 k1), k3 = f(n + dt/2 k2), k4 = f(n + dt k3),
 * n <- n + dt/6 (k1 + 2 k2 + 2 k3 + k4), renormalised every step ("all [Runge-Kutta methods] have this property", :367).
 * The stage configurations are not renormalised; the thermal field of the step is the same in all four stages (R11).    */
static void orc_rk4_step(orc_system *s) {
    long N = s->N; int nb = s->nb; (void)nb;
    double *F = (double *)malloc(3 * N * sizeof(double)), *y = (double *)malloc(3 * N * sizeof(double));
    double *acc = (double *)calloc(3 * N, sizeof(double)), *sg = (double *)calloc(3 * N, sizeof(double)), *Fth = NULL;
    if (s->T > 0.0) {
        Fth = (double *)malloc(3 * N * sizeof(double));
        for (long i = 0; i < N; ++i) {
            double xi[3]; orc_thermal_xi_image(s->seed, s->step, (uint32_t)i, s->image, xi);
            double sig = thermal_sigma_site(s, i);
            for (int k = 0; k < 3; ++k) Fth[3*i+k] = sig * xi[k];
        }
    }
    const double cnext[4] = { 0.5, 0.5, 1.0, 0.0 }, wacc[4] = { 1.0, 2.0, 2.0, 1.0 };
    memcpy(y, s->n, 3 * N * sizeof(double));
    for (int st = 0; st < 4; ++st) {
        total_force(s, y, Fth, F);
        if (s->u != 0.0) orc_stt_gradient(s, y, sg);
        for (long i = 0; i < N; ++i) {
            double A[3], k[3];
            rot_field(s, i, y + 3*i, F + 3*i, sg + 3*i, A);
            cross3(y + 3*i, A, k);
            for (int c = 0; c < 3; ++c) acc[3*i+c] += wacc[st] * k[c];
            if (s->pinned && s->pinned[i]) continue;
            if (st < 3) for (int c = 0; c < 3; ++c) y[3*i+c] = s->n[3*i+c] + cnext[st] * s->dt * k[c];
        }
    }
    for (long i = 0; i < N; ++i) {
        if (s->pinned && s->pinned[i]) continue;
        double out[3];
        for (int c = 0; c < 3; ++c) out[c] = s->n[3*i+c] + s->dt / 6.0 * acc[3*i+c];
        double nrm = sqrt(dot3(out, out));
        for (int c = 0; c < 3; ++c) s->n[3*i+c] = out[c] / nrm;
    }
    s->step += 1;
    free(F); free(y); free(acc); free(sg); free(Fth);
}
void orc_llg_iterate(orc_system *s, long nsteps) { for (long k = 0; k < nsteps; ++k) orc_llg_step(s); }

/* Heun's method, B3-B4 with f = n x A, renormalised every step.  Only used to pin Fig. 5's
 * "Heun within 1e-6 / Depondt 3e-7" statement; no thermal field, no current.                */
void orc_heun_step(orc_system *s) {
    long N = s->N; int nb = s->nb; (void)nb;
    double *F = (double *)malloc(3 * N * sizeof(double)), *f0 = (double *)malloc(3 * N * sizeof(double));
    double *np_ = (double *)malloc(3 * N * sizeof(double)), *sg = (double *)calloc(3 * N, sizeof(double));
    total_force(s, s->n, NULL, F);
    for (long i = 0; i < N; ++i) {
        double A[3]; rot_field(s, i, s->n + 3*i, F + 3*i, sg + 3*i, A);
        cross3(s->n + 3*i, A, f0 + 3*i);
        for (int k = 0; k < 3; ++k) np_[3*i+k] = s->n[3*i+k] + s->dt * f0[3*i+k];
    }
    total_force(s, np_, NULL, F);
    for (long i = 0; i < N; ++i) {
        double A[3], f1[3], out[3];
        rot_field(s, i, np_ + 3*i, F + 3*i, sg + 3*i, A);
        cross3(np_ + 3*i, A, f1);
        for (int k = 0; k < 3; ++k) out[k] = s->n[3*i+k] + 0.5 * s->dt * (f0[3*i+k] + f1[k]);
        double nrm = sqrt(dot3(out, out));
        for (int k = 0; k < 3; ++k) s->n[3*i+k] = out[k] / nrm;
    }
    s->step += 1;
    free(F); free(f0); free(np_); free(sg);
}

/* ------------------------------------------------------------------ velocity-projection minimiser, App. D (:438-463)
 * "Pretend that the spins are massive particles moving on the surfaces of spheres", force F_i = -dH/dn_i (D4).  One iteration,
 * in the order the appendix lists the equations (reading R28: the paper does not say where in the step the force is evaluated):
 *     F(t+dt) = F(x(t))                                  force of the current configuration            (D4)
 *     v <- v + dt/(2m) (F(t) + F(t+dt))                  velocity increment                             (D2)
 *     v <- (v.F) F/|F|^2 if v.F > 0 else 0               projection, dot products over all 3N components (D3)
 *     x <- x + dt v + dt^2/(2m) F                        position increment                             (D1)
 *     x_i <- x_i/|x_i|                                   renormalisation                                (D5)
 * The first iteration starts from v = 0 and F(t) = F(t+dt).  Pinned spins do not move and carry no force.            */
void orc_vp_reset(orc_system *s) { free(s->vp_v); free(s->vp_F); s->vp_v = NULL; s->vp_F = NULL; }
void orc_vp_iterate(orc_system *s, long n_iter, double dt, double mass) {
    long N = s->N; int nb = s->nb; (void)nb;
    double *F = (double *)malloc(3 * N * sizeof(double));
    for (long it = 0; it < n_iter; ++it) {
        orc_gradient(s, s->n, F, T_ALL);
        if (s->pinned) for (long i = 0; i < N; ++i) if (s->pinned[i]) { F[3*i] = 0; F[3*i+1] = 0; F[3*i+2] = 0; }
        if (!s->vp_v) {
            s->vp_v = (double *)calloc(3 * N, sizeof(double));
            s->vp_F = (double *)malloc(3 * N * sizeof(double));
            memcpy(s->vp_F, F, 3 * N * sizeof(double));
        }
        long double vF = 0.0L, FF = 0.0L;
        for (long i = 0; i < 3 * N; ++i) {
            s->vp_v[i] += 0.5 * dt / mass * (s->vp_F[i] + F[i]);                          /* D2 */
            vF += (long double)s->vp_v[i] * F[i];
            FF += (long double)F[i] * F[i];
        }
        double ratio = (vF > 0.0L && FF > 0.0L) ? (double)(vF / FF) : 0.0;                /* D3 */
        for (long i = 0; i < N; ++i) {
            if (s->pinned && s->pinned[i]) { for (int k = 0; k < 3; ++k) s->vp_v[3*i+k] = 0.0; continue; }
            double x[3];
            for (int k = 0; k < 3; ++k) {
                s->vp_v[3*i+k] = ratio * F[3*i+k];
                x[k] = s->n[3*i+k] + dt * s->vp_v[3*i+k] + 0.5 * dt * dt / mass * F[3*i+k];   /* D1 */
            }
            double nrm = sqrt(dot3(x, x));
            for (int k = 0; k < 3; ++k) s->n[3*i+k] = x[k] / nrm;                          /* D5 */
        }
        memcpy(s->vp_F, F, 3 * N * sizeof(double));
    }
    free(F);
}

/* ------------------------------------------------------------------ geodesic nudged elastic band, III.D (:193-216) and App. F
 * A chain of M images (configurations) of the same system; chain[nu] points at 3N doubles.  One call computes, for every
 * interior image, the total force of Eq. 14, F = F^S + F^E (3N-dimensional vectors):
 *   tangent      "the definitions given in Ref. 55" (:212; Henkelman-Jonsson): tau+ = n_{nu+1} - n_nu, tau- = n_nu - n_{nu-1};
 *                tau = tau+ if E_{nu+1} > E_nu > E_{nu-1}; tau- if E_{nu+1} < E_nu < E_{nu-1}; otherwise the mix
 *                tau+ dEmax + tau- dEmin (E_{nu+1} > E_{nu-1}) or tau+ dEmin + tau- dEmax, dEmax/min = max/min |E_{nu+-1} - E_nu|;
 *                then projected on the tangent space of the image, spin by spin (F1), and normalised in 3N dimensions
 *   distance     l_{nu,mu}: geodesic, sqrt(sum_i angle(n_{nu,i}, n_{mu,i})^2) (:477 "the great-circle distance")
 *   spring       F^S = kappa (l_{nu,nu+1} - l_{nu-1,nu}) tau (Eq. 15; the printed order of the two lengths would push an image
 *                towards its nearer neighbour and bunch the chain up -- reading R31; kappa = 1 in the paper)
 *   gradient     F^E = -grad E + (grad E . tau) tau (Eq. 16); climbing image: F^S = 0, F^E = -grad E + 2 (grad E . tau) tau (Eq. 17);
 *                the total is projected on the tangent space spin by spin (F2)
 * End images get zero force.  E_out[nu] receives the energies, l_out[nu] = l_{nu,nu+1}.  F_out: M x 3N.                  */
static double geodesic_distance(long N, const double *a, const double *b) {
    long double s2 = 0.0L;
    for (long i = 0; i < N; ++i) {
        double c[3]; cross3(a + 3*i, b + 3*i, c);
        double ang = atan2(sqrt(dot3(c, c)), dot3(a + 3*i, b + 3*i));
        s2 += (long double)ang * ang;
    }
    return (double)sqrtl(s2);
}
double orc_geodesic_distance(const orc_system *s, const double *a, const double *b) { return geodesic_distance(s->N, a, b); }
void orc_gneb_forces(orc_system *s, int M, const double *chain, double kappa, int climbing, double *F_out, double *E_out, double *l_out) {
    long N = s->N; int nb = s->nb; (void)nb;
    double *E = (double *)malloc(M * sizeof(double)), *l = (double *)calloc(M, sizeof(double));
    double *G = (double *)malloc(3 * N * sizeof(double)), *tau = (double *)malloc(3 * N * sizeof(double));
    for (int nu = 0; nu < M; ++nu) {
        double Et[6]; orc_energy(s, chain + (size_t)nu * 3 * N, Et);
        E[nu] = Et[0] + Et[1] + Et[2] + Et[3] + Et[4] + Et[5];
        if (nu + 1 < M) l[nu] = geodesic_distance(N, chain + (size_t)nu * 3 * N, chain + (size_t)(nu + 1) * 3 * N);
    }
    memset(F_out, 0, (size_t)M * 3 * N * sizeof(double));
    for (int nu = 1; nu + 1 < M; ++nu) {
        const double *n = chain + (size_t)nu * 3 * N, *np_ = chain + (size_t)(nu + 1) * 3 * N, *nm = chain + (size_t)(nu - 1) * 3 * N;
        double wp, wm;                                    /* tau = wp tau+ + wm tau- */
        if (E[nu + 1] > E[nu] && E[nu] > E[nu - 1]) { wp = 1.0; wm = 0.0; }
        else if (E[nu + 1] < E[nu] && E[nu] < E[nu - 1]) { wp = 0.0; wm = 1.0; }
        else {
            double dp = fabs(E[nu + 1] - E[nu]), dm = fabs(E[nu - 1] - E[nu]);
            double dmax = dp > dm ? dp : dm, dmin = dp > dm ? dm : dp;
            if (E[nu + 1] > E[nu - 1]) { wp = dmax; wm = dmin; } else { wp = dmin; wm = dmax; }
            if (wp == 0.0 && wm == 0.0) { wp = 1.0; wm = 1.0; }      /* flat energy: the central difference */
        }
        long double t2 = 0.0L;
        for (long i = 0; i < N; ++i) {
            double t[3];
            for (int k = 0; k < 3; ++k) t[k] = wp * (np_[3*i+k] - n[3*i+k]) + wm * (n[3*i+k] - nm[3*i+k]);
            double p = dot3(t, n + 3*i);
            for (int k = 0; k < 3; ++k) { tau[3*i+k] = t[k] - p * n[3*i+k]; t2 += (long double)tau[3*i+k] * tau[3*i+k]; }   /* F1 */
        }
        double tn = (double)sqrtl(t2);
        for (long i = 0; i < 3 * N; ++i) tau[i] = tn > 0.0 ? tau[i] / tn : 0.0;
        orc_gradient(s, n, G, T_ALL);                     /* G = -grad E */
        if (s->pinned) for (long i = 0; i < N; ++i) if (s->pinned[i]) { G[3*i] = 0; G[3*i+1] = 0; G[3*i+2] = 0; }
        long double gt = 0.0L;
        for (long i = 0; i < 3 * N; ++i) gt += (long double)G[i] * tau[i];
        double *F = F_out + (size_t)nu * 3 * N;
        double cs = (nu == climbing) ? 0.0 : kappa * (l[nu] - l[nu - 1]);       /* Eq. 15 / 17 */
        double ce = (nu == climbing) ? 2.0 * (double)gt : (double)gt;           /* Eq. 16 / 17: G - (G.tau) tau */
        for (long i = 0; i < N; ++i) {
            double f[3];
            for (int k = 0; k < 3; ++k) f[k] = G[3*i+k] - ce * tau[3*i+k] + cs * tau[3*i+k];
            double p = dot3(f, n + 3*i);
            for (int k = 0; k < 3; ++k) F[3*i+k] = (s->pinned && s->pinned[i]) ? 0.0 : f[k] - p * n[3*i+k];             /* F2 */
        }
    }
    if (E_out) memcpy(E_out, E, M * sizeof(double));
    if (l_out) memcpy(l_out, l, M * sizeof(double));
    free(E); free(l); free(G); free(tau);
}
/* one relaxation step of the chain: x <- x + step F, renormalised (plain steepest descent; the paper does not fix the optimiser) */
void orc_gneb_iterate(orc_system *s, int M, double *chain, long n_iter, double step, double kappa, int climbing) {
    long N = s->N; int nb = s->nb; (void)nb;
    double *F = (double *)malloc((size_t)M * 3 * N * sizeof(double));
    for (long it = 0; it < n_iter; ++it) {
        orc_gneb_forces(s, M, chain, kappa, climbing, F, NULL, NULL);
        for (int nu = 1; nu + 1 < M; ++nu)
            for (long i = 0; i < N; ++i) {
                double *x = chain + (size_t)nu * 3 * N + 3 * i, *f = F + (size_t)nu * 3 * N + 3 * i, y[3];
                if (s->pinned && s->pinned[i]) continue;
                for (int k = 0; k < 3; ++k) y[k] = x[k] + step * f[k];
                double nrm = sqrt(dot3(y, y));
                for (int k = 0; k < 3; ++k) x[k] = y[k] / nrm;
            }
    }
    free(F);
}

/* ------------------------------------------------------------------ topological charge, App. A (:317-343)
 * Q = (1/4 pi) sum_l A_l (A1) over the elementary triangles l of every a-b plane, A_l the signed area of the spherical
 * triangle (n_i, n_j, n_k):  cos(A_l/2) = (1 + ni.nj + ni.nk + nj.nk) / sqrt(2 (1+ni.nj)(1+nj.nk)(1+nk.ni))  (A2),
 * sign(A_l) = sign[n_i . (n_j x n_k)] (the extracted text prints "n_i . (n_i x n_k)", which is identically zero: garbled,
 * reading R26).  Triangles: each cell (ia, ib) gives (r, r+a, r+a+b) and (r, r+a+b, r+b), counter-clockwise about +z
 * when (a x b).z > 0 (the order is mirrored otherwise, :331).  One basis atom.  A triangle with a corner outside an open
 * edge is skipped; periodic directions wrap (":343 only defined with periodical boundary conditions").               */
static double spherical_area(const double *ni, const double *nj, const double *nk) {
    double ij = dot3(ni, nj), ik = dot3(ni, nk), jk = dot3(nj, nk);
    double den = sqrt(2.0 * (1.0 + ij) * (1.0 + jk) * (1.0 + ik));
    if (den == 0.0) return 0.0;                        /* exceptional configuration (A3): not defined, counted as 0 */
    double c = (1.0 + ij + ik + jk) / den;
    if (c > 1.0) c = 1.0;
    if (c < -1.0) c = -1.0;
    double A = 2.0 * acos(c), jxk[3];
    cross3(nj, nk, jxk);
    double t = dot3(ni, jxk);
    return t > 0.0 ? A : (t < 0.0 ? -A : 0.0);
}
double orc_spherical_area(const double *ni, const double *nj, const double *nk) { return spherical_area(ni, nj, nk); }
double orc_topological_charge(const orc_system *s, const double *n) {
    if (s->nb != 1) return NAN;
    const double *a = s->brav, *b = s->brav + 3;
    int ccw = (a[0] * b[1] - a[1] * b[0]) > 0.0;
    long double sum = 0.0L;
    for (int ic = 0; ic < s->nc[2]; ++ic)
        for (int ib = 0; ib < s->nc[1]; ++ib)
            for (int ia = 0; ia < s->nc[0]; ++ia) {
                int ia1 = ia + 1, ib1 = ib + 1;
                if (ia1 == s->nc[0]) { if (!s->per[0]) continue; ia1 = 0; }
                if (ib1 == s->nc[1]) { if (!s->per[1]) continue; ib1 = 0; }
                int c00[3] = {ia, ib, ic}, c10[3] = {ia1, ib, ic}, c11[3] = {ia1, ib1, ic}, c01[3] = {ia, ib1, ic};
                const double *n00 = n + 3 * cell_index(s, c00), *n10 = n + 3 * cell_index(s, c10);
                const double *n11 = n + 3 * cell_index(s, c11), *n01 = n + 3 * cell_index(s, c01);
                if (ccw) sum += spherical_area(n00, n10, n11) + spherical_area(n00, n11, n01);
                else     sum += spherical_area(n00, n11, n10) + spherical_area(n00, n01, n11);
            }
    return (double)(sum / (4.0L * (long double)ORC_PI));
}

/* ------------------------------------------------------------------ what the boundary returns
 * effective_field: deterministic F/(mu_s mu_B) in Tesla (reading R2).
 * observables: M = (1/N) sum n_i (:131) and max_i |F_i - (F_i.n_i) n_i| in meV (reading R22). */
void orc_effective_field(orc_system *s, double *B) {
    orc_gradient(s, s->n, B, T_ALL);
    for (long i = 0; i < s->N; ++i) {
        double m = mu_at(s, i) * ORC_MU_B;
        for (int k = 0; k < 3; ++k) B[3*i+k] /= m;
    }
}
void orc_observables(orc_system *s, double M[3], double *max_torque) {
    double *F = (double *)malloc(3 * s->N * sizeof(double));
    orc_gradient(s, s->n, F, T_ALL);
    long double m[3] = {0, 0, 0}; double mt = 0.0;
    for (long i = 0; i < s->N; ++i) {
        const double *n = s->n + 3*i; double p = dot3(F + 3*i, n), t[3];
        for (int k = 0; k < 3; ++k) { m[k] += n[k]; t[k] = F[3*i+k] - p * n[k]; }
        double tn = sqrt(dot3(t, t));
        if (s->pinned && s->pinned[i]) continue;           /* a pinned spin carries no torque that matters */
        if (tn > mt) mt = tn;
    }
    for (int k = 0; k < 3; ++k) M[k] = (double)(m[k] / (long double)s->N);
    *max_torque = mt;
    free(F);
}
