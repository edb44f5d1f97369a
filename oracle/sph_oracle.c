/*
 * sph_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the SPH hot path computes (density sum with
 * smoothing-length iteration, then the symmetric hydro-force pair sum).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call it.  It shares no code, header, table or helper with the CUDA path in
 * paper_2003_10850_b200/csrc and neither includes the other.
 *
 * Authority.  The paper states the problem only: "computes particle densities by
 * multiple iterations and the second one computes hydrodynamic forces" (§1), for
 * a list of active particles "find all neighbouring particles within a given distance"
 * (§1); the SPH formulation is delegated to its refs [2] and [6] (§1).
 * Every formula below is therefore a READING, restated from that published lineage and listed
 * in DESIGN.md §"Readings" (R1..R16, following SURVEY.md §8(c)); the section tags in the
 * comments name the reading.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): kernel normalisation integral = 1 and
 * central values 8/pi, 1365/(64 pi); finite-difference derivative identities; equal-mass
 * identity N_w = (4 pi/3) H^3 rho/m; perfect-lattice values; two-particle hand computation;
 * brute force == cell list; momentum and energy conservation; viscous heating >= 0; static gas
 * v_sig = 2 sqrt(gamma (gamma-1) u); permutation / translation / axis-swap / scaling symmetries;
 * the sums S, D', rho, d rho/dH and Omega of an evaluation against centred finite differences of
 * S(H) and rho(H); the R7 step: exact landing on the root of a power-law medium whose logarithmic
 * slope is not 3 (pins the slope factor g and the logarithmic Newton step), the clamp 2^(-1/3) as a
 * closed form, and a constructed integer-count case with the closed-form trajectory
 * clamp, clamp, clamp, bracket, 19 volume bisections hi_k^3 = 1 + 2^-k, BRACKET flag
 * (pins the bracket, the strict r < H, the bisection and the collapse rule); the edge-class flags are
 * bounded (<= 2 % of a config-1 set).
 * PARITY UNPINNED BY THE PAPER: which H inside the tolerance band is returned follows from the rule
 * R7 written here (the paper says only "multiple iterations"); R7 is FROZEN since round 2:
 * tests/golden/h_trajectory.txt (written by tests/golden/make_h_trajectory.py from this file alone)
 * holds the trajectories of a seeded set, and any change to the rule must come with a new pin and a
 * DESIGN.md reading.
 *
 * Summation order: ascending j inside a cell, cells in ascending index order; brute force in
 * ascending j.  No blocking, fusion or reordering beyond the definitions.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int kernel;      /* 0 cubic spline, 1 Wendland C6 (R1) */
    double box;      /* periodic cube edge L */
    double gamma;    /* adiabatic index */
    double alpha;    /* artificial viscosity alpha (R9) */
    int count_mode;  /* 0: kernel-weighted number N_w drives the iteration, 1: integer count (R2) */
    int max_iter;    /* iteration cap (R7) */
} orc_params;

/* flags returned per particle by orc_density */
#define ORC_F_CONVERGED 1
#define ORC_F_BRACKET 2   /* bracket collapsed */
#define ORC_F_NOTCONV 4   /* max_iter reached */
#define ORC_F_STALLED 8   /* update could not move H (cap at 0.49999 L) */
/* edge-class bits: the fp32 path may legitimately take the other branch */
#define ORC_E_RADIUS 1    /* some neighbour with |r/H - 1| < 1e-6 at some evaluation */
#define ORC_E_BAND 2      /* | |N-N_t| - tol | < 1e-4 N_t at some evaluation */
#define ORC_E_BRANCH 4    /* clamp / bisection / slope guard within 1e-6 of switching */

/* ---------------------------------------------------------------- kernels (R1, R3, R4) */
/* W(r,H) = sigma H^-3 w(q), q = r/H, H = support radius (W = 0 for q >= 1). */
static double k_sigma(int k) { return k == 0 ? 8.0 / M_PI : 1365.0 / (64.0 * M_PI); }

static double k_w(int k, double q)
{
    if (q >= 1.0) return 0.0;
    if (k == 0) {
        if (q <= 0.5) return 1.0 - 6.0 * q * q + 6.0 * q * q * q;
        double t = 1.0 - q;
        return 2.0 * t * t * t;
    } else {
        double t = 1.0 - q;
        double t2 = t * t, t4 = t2 * t2, t8 = t4 * t4;
        return t8 * (1.0 + 8.0 * q + 25.0 * q * q + 32.0 * q * q * q);
    }
}

static double k_dw(int k, double q) /* w'(q) */
{
    if (q >= 1.0) return 0.0;
    if (k == 0) {
        if (q <= 0.5) return -12.0 * q + 18.0 * q * q;
        double t = 1.0 - q;
        return -6.0 * t * t;
    } else {
        double t = 1.0 - q;
        double t2 = t * t, t4 = t2 * t2, t7 = t4 * t2 * t;
        return -22.0 * q * t7 * (1.0 + 7.0 * q + 16.0 * q * q);
    }
}

/* exported so the pins can integrate / differentiate them */
double orc_kernel_w(int k, double q) { return k_w(k, q); }
double orc_kernel_dw(int k, double q) { return k_dw(k, q); }
double orc_kernel_sigma(int k) { return k_sigma(k); }
double orc_W(int k, double r, double H) { return k_sigma(k) / (H * H * H) * k_w(k, r / H); }
double orc_dWdr(int k, double r, double H) { return k_sigma(k) / (H * H * H * H) * k_dw(k, r / H); }
double orc_dWdH(int k, double r, double H)
{
    double q = r / H;
    return -k_sigma(k) / (H * H * H * H) * (3.0 * k_w(k, q) + q * k_dw(k, q));
}

/* ---------------------------------------------------------------- geometry (R11: static periodic box) */
static inline double min_image(double d, double L)
{
    if (d >= 0.5 * L) d -= L;
    else if (d < -0.5 * L) d += L;
    return d;
}

/* uniform periodic grid; used only to skip cells that cannot hold a neighbour */
typedef struct {
    int G;
    double L;
    int64_t *start; /* G^3 + 1 */
    int32_t *idx;   /* particle ids, ascending inside a cell */
    double *hmax;   /* per-cell max support radius (force pass), may be NULL */
} orc_grid;

static inline int cell_of(const orc_grid *g, double x)
{
    int c = (int)floor(x / g->L * g->G);
    if (c < 0) c = 0;
    if (c >= g->G) c = g->G - 1;
    return c;
}

static orc_grid *grid_build(int64_t n, const float *pos, double L, double cell_hint, const float *h)
{
    orc_grid *g = (orc_grid *)calloc(1, sizeof(orc_grid));
    int G = (int)floor(L / (cell_hint > 0 ? cell_hint : L));
    if (G < 1) G = 1;
    if (G > 160) G = 160;
    g->G = G;
    g->L = L;
    int64_t nc = (int64_t)G * G * G;
    g->start = (int64_t *)calloc(nc + 1, sizeof(int64_t));
    g->idx = (int32_t *)malloc(sizeof(int32_t) * (n > 0 ? n : 1));
    g->hmax = h ? (double *)calloc(nc, sizeof(double)) : NULL;
    int64_t *cnt = (int64_t *)calloc(nc, sizeof(int64_t));
    for (int64_t i = 0; i < n; i++) {
        int64_t c = ((int64_t)cell_of(g, pos[3 * i + 2]) * G + cell_of(g, pos[3 * i + 1])) * G + cell_of(g, pos[3 * i]);
        cnt[c]++;
        if (h && (double)h[i] > g->hmax[c]) g->hmax[c] = (double)h[i];
    }
    for (int64_t c = 0; c < nc; c++) g->start[c + 1] = g->start[c] + cnt[c];
    memset(cnt, 0, sizeof(int64_t) * nc);
    for (int64_t i = 0; i < n; i++) {
        int64_t c = ((int64_t)cell_of(g, pos[3 * i + 2]) * G + cell_of(g, pos[3 * i + 1])) * G + cell_of(g, pos[3 * i]);
        g->idx[g->start[c] + cnt[c]++] = (int32_t)i;
    }
    free(cnt);
    return g;
}

static void grid_free(orc_grid *g)
{
    if (!g) return;
    free(g->start);
    free(g->idx);
    free(g->hmax);
    free(g);
}

/* cells of one axis that can hold a point within R of x: [lo, lo+cnt) modulo G, each at most once */
static void axis_range(const orc_grid *g, double x, double R, int *lo, int *cnt)
{
    double cs = g->L / g->G;
    int a = (int)floor((x - R) / cs) - 1; /* one cell of slack: pruning only, never correctness */
    int b = (int)floor((x + R) / cs) + 1;
    int c = b - a + 1;
    if (c >= g->G) { *lo = 0; *cnt = g->G; }
    else { *lo = a; *cnt = c; }
}

/* minimum distance^2 from point to a cell (periodic), lower bound used for pruning */
static double cell_mindist2(const orc_grid *g, const double *x, int cx, int cy, int cz)
{
    double cs = g->L / g->G, s = 0.0;
    int c[3] = {cx, cy, cz};
    for (int a = 0; a < 3; a++) {
        double centre = (c[a] + 0.5) * cs;
        double d = fabs(min_image(x[a] - centre, g->L)) - 0.5 * cs;
        if (d > 0) s += d * d;
    }
    return s;
}

/* ---------------------------------------------------------------- density (R1-R6, R13) */
typedef struct {
    double S;      /* sum_j W(r_ij, H)                       */
    double Dp;     /* sum_j dW/dH(r_ij, H)                   */
    double rho;    /* sum_j m_j W                            */
    double drho;   /* sum_j m_j dW/dH                        */
    double Nw;     /* (4 pi/3) H^3 S                         */
    int32_t Nint;  /* #{j : r_ij < H}, self included, strict */
    int edge;      /* some j with |r/H - 1| < 1e-6           */
} dens_eval;

typedef struct {
    const orc_params *p;
    int64_t n;
    const float *pos;
    const float *mass; /* NULL -> mass_scalar */
    double mass_scalar;
    const orc_grid *grid; /* NULL -> brute force over all j */
} dens_ctx;

static inline void dens_pair(const dens_ctx *c, const double *xi, double H, int64_t j, dens_eval *e)
{
    double L = c->p->box;
    double dx = min_image(xi[0] - (double)c->pos[3 * j], L);
    double dy = min_image(xi[1] - (double)c->pos[3 * j + 1], L);
    double dz = min_image(xi[2] - (double)c->pos[3 * j + 2], L);
    double r2 = dx * dx + dy * dy + dz * dz;
    double r = sqrt(r2);
    if (fabs(r / H - 1.0) < 1e-6) e->edge = 1;
    if (!(r2 < H * H)) return; /* strict (R4) */
    double mj = c->mass ? (double)c->mass[j] : c->mass_scalar;
    double W = orc_W(c->p->kernel, r, H);       /* the pinned kernel functions themselves (R1) */
    double dWdH = orc_dWdH(c->p->kernel, r, H);
    e->S += W;
    e->Dp += dWdH;
    e->rho += mj * W;
    e->drho += mj * dWdH;
    e->Nint += 1;
}

static void dens_at(const dens_ctx *c, int64_t i, double H, dens_eval *e)
{
    memset(e, 0, sizeof(*e));
    double xi[3] = {(double)c->pos[3 * i], (double)c->pos[3 * i + 1], (double)c->pos[3 * i + 2]};
    if (!c->grid) {
        for (int64_t j = 0; j < c->n; j++) dens_pair(c, xi, H, j, e); /* self term j = i included (R5) */
    } else {
        const orc_grid *g = c->grid;
        int lo[3], cnt[3];
        for (int a = 0; a < 3; a++) axis_range(g, xi[a], H * (1.0 + 2e-6), &lo[a], &cnt[a]);
        for (int kz = 0; kz < cnt[2]; kz++)
            for (int ky = 0; ky < cnt[1]; ky++)
                for (int kx = 0; kx < cnt[0]; kx++) {
                    int cx = ((lo[0] + kx) % g->G + g->G) % g->G;
                    int cy = ((lo[1] + ky) % g->G + g->G) % g->G;
                    int cz = ((lo[2] + kz) % g->G + g->G) % g->G;
                    int64_t cc = ((int64_t)cz * g->G + cy) * g->G + cx;
                    for (int64_t s = g->start[cc]; s < g->start[cc + 1]; s++) dens_pair(c, xi, H, g->idx[s], e);
                }
    }
    e->Nw = 4.0 * M_PI / 3.0 * H * H * H * e->S;
}

/* One evaluation at the given support radii (h[i], fp32 input promoted) for the listed particles. */
int orc_density_eval(const orc_params *p, int64_t n, const float *pos, const float *mass, double mass_scalar,
                     const float *h, const int32_t *active, int64_t n_active, int brute, double cell_hint,
                     double *S, double *Dp, double *rho, double *drho, double *Nw, int32_t *Nint, uint8_t *edge)
{
    orc_grid *g = brute ? NULL : grid_build(n, pos, p->box, cell_hint, NULL);
    dens_ctx c = {p, n, pos, mass, mass_scalar, g};
    int64_t na = active ? n_active : n;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        dens_eval e;
        dens_at(&c, i, (double)h[i], &e);
        S[a] = e.S; Dp[a] = e.Dp; rho[a] = e.rho; drho[a] = e.drho; Nw[a] = e.Nw; Nint[a] = e.Nint;
        if (edge) edge[a] = (uint8_t)(e.edge ? ORC_E_RADIUS : 0);
    }
    grid_free(g);
    return 0;
}

/*
 * The h iteration (R7; "computes particle densities by multiple iterations", §1).
 * Per active particle, independently: safeguarded Newton iteration on the neighbour number in
 * logarithmic variables, F(x) = ln N_w(e^x) - ln N_t with x = ln H.  Since
 *   N_w = (4 pi/3) H^3 S(H),   d ln N_w / d ln H = 3 (1 + H S'/(3 S)) = 3 / g,   g = 1/(1 + H D'/(3 S)),
 * the Newton step x - F/F' is  H <- H (N_t / N_w)^(g/3).  (N_w is locally a power law of H -- exactly
 * H^3 in a uniform medium, where this step lands on the root at once; the same Newton step taken on
 * N_w(H) directly, H [1 - (N_w - N_t)/(3 N_w) g], needs 20 % more evaluations on the clustered sets.)
 * With count_mode 1 the integer count N_int replaces N_w in the same expressions.
 */
int orc_density(const orc_params *p, int64_t n, const float *pos, const float *mass, double mass_scalar,
                const float *h_guess, const int32_t *active, int64_t n_active, double n_target, double n_tol,
                int brute, double cell_hint,
                double *H_out, double *rho, double *omega, double *Nw_out, int32_t *Nint, int32_t *iters,
                int32_t *flags, uint8_t *edge, int64_t *n_evals_total)
{
    orc_grid *g = brute ? NULL : grid_build(n, pos, p->box, cell_hint, NULL);
    dens_ctx c = {p, n, pos, mass, mass_scalar, g};
    int64_t na = active ? n_active : n;
    const double smin = pow(2.0, -1.0 / 3.0), smax = pow(2.0, 1.0 / 3.0);
    const double Hcap = 0.49999 * p->box;
    int64_t evals = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : evals)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        double H = (double)h_guess[i], lo = 0.0, hi = INFINITY;
        int it = 0, flag = 0, eb = 0;
        dens_eval e;
        for (;;) {
            dens_at(&c, i, H, &e);
            it++;
            evals++;
            if (e.edge) eb |= ORC_E_RADIUS;
            double N = p->count_mode ? (double)e.Nint : e.Nw;
            double dev = fabs(N - n_target);
            if (isfinite(n_tol) && fabs(dev - n_tol) < 1e-4 * n_target) eb |= ORC_E_BAND;
            if (dev <= n_tol) { flag = ORC_F_CONVERGED; break; } /* inclusive */
            if (it >= p->max_iter) { flag = ORC_F_NOTCONV; break; }
            if (N < n_target) { if (H > lo) lo = H; } else { if (H < hi) hi = H; }
            if (isfinite(hi) && lo > 0.0) {
                if (fabs((hi - lo) - 1e-6 * lo) < 1e-9 * lo) eb |= ORC_E_BRANCH;
                if (hi - lo <= 1e-6 * lo) { flag = ORC_F_BRACKET; break; }
            }
            double gsl = 1.0 / (1.0 + H * e.Dp / (3.0 * e.S));
            if (fabs(gsl) < 1e-6 || fabs(gsl - 4.0) < 1e-6) eb |= ORC_E_BRANCH;
            if (!(gsl > 0.0 && gsl < 4.0) || N == 0.0) gsl = 1.0;
            double s = (N == 0.0) ? smax : pow(n_target / N, gsl / 3.0);
            if (fabs(s - smin) < 1e-6 || fabs(s - smax) < 1e-6) eb |= ORC_E_BRANCH;
            if (s < smin) s = smin;
            if (s > smax) s = smax;
            double Hn = H * s;
            if (isfinite(hi) && lo > 0.0) {
                if (fabs(Hn - lo) < 1e-6 * lo || fabs(Hn - hi) < 1e-6 * hi) eb |= ORC_E_BRANCH;
                if (!(lo < Hn && Hn < hi)) Hn = cbrt(0.5 * (lo * lo * lo + hi * hi * hi)); /* volume bisection */
            }
            if (Hn > Hcap) Hn = Hcap;
            if (Hn == H) { flag = ORC_F_STALLED; break; }
            H = Hn;
        }
        H_out[a] = H;
        rho[a] = e.rho;
        omega[a] = 1.0 + H / (3.0 * e.rho) * e.drho; /* grad-h factor Omega (R1) */
        Nw_out[a] = e.Nw;
        Nint[a] = e.Nint;
        iters[a] = it;
        flags[a] = flag;
        if (edge) edge[a] = (uint8_t)eb;
    }
    if (n_evals_total) *n_evals_total = evals;
    grid_free(g);
    return 0;
}

/* ---------------------------------------------------------------- hydro force (R8-R12) */
/*
 * For every active i, over all j != i with r_ij < max(H_i, H_j):
 *   F_ij(H) = dW/dr(r_ij, H) (0 for r >= H), rhat = d_ij / r, v_ij = v_i - v_j,
 *   mu = min(0, v_ij.rhat), v_sig,ij = c_i + c_j - 3 mu, Pi = -(alpha/2) v_sig mu / rhobar,
 *   Fbar = (F_ij(H_i) + F_ij(H_j))/2,  A_k = P_k / (Omega_k rho_k^2), P = (gamma-1) rho u,
 *   a_i     = - sum_j m_j [A_i F_ij(H_i) + A_j F_ij(H_j) + Pi Fbar] rhat
 *   du_i/dt =   sum_j m_j [A_i F_ij(H_i) + Pi Fbar / 2] (v_ij.rhat)
 *   vsig_i  =   max_j v_sig,ij   (0 if the set is empty)
 * Coincident pairs (r = 0, j != i) give nothing to a, du/dt and c_i + c_j to vsig.
 * Inactive neighbours enter with their current (h, rho, Omega, u, v) (R12).
 */
typedef struct {
    double a[3], du, vsig;
    double asum, dusum; /* sums of |pair term| for the parity tolerance floor (R15) */
    double asq, dusq;   /* sums of (pair term)^2: the fp32 resolution of the sum (R15), test-side only */
    double duvisc;      /* viscous part of du/dt (pin: >= 0) */
    int64_t npair;
    int edge;
} force_acc;

typedef struct {
    const orc_params *p;
    int64_t n;
    const float *pos, *vel, *u, *mass, *h, *rho, *omega;
    double mass_scalar;
} force_ctx;

static inline void force_pair(const force_ctx *c, int64_t i, int64_t j, force_acc *f)
{
    if (j == i) return;
    const orc_params *p = c->p;
    double L = p->box;
    double d[3];
    for (int a = 0; a < 3; a++) d[a] = min_image((double)c->pos[3 * i + a] - (double)c->pos[3 * j + a], L);
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double Hi = (double)c->h[i], Hj = (double)c->h[j];
    double Hm = Hi > Hj ? Hi : Hj;
    double r = sqrt(r2);
    if (fabs(r / Hm - 1.0) < 1e-6) f->edge = 1;
    if (!(r2 < Hm * Hm)) return;
    double gm1 = p->gamma - 1.0;
    double ci = sqrt(p->gamma * gm1 * (double)c->u[i]), cj = sqrt(p->gamma * gm1 * (double)c->u[j]);
    f->npair++;
    if (r == 0.0) {
        if (ci + cj > f->vsig) f->vsig = ci + cj;
        return;
    }
    double rhoi = (double)c->rho[i], rhoj = (double)c->rho[j];
    double Ai = gm1 * (double)c->u[i] / ((double)c->omega[i] * rhoi);
    double Aj = gm1 * (double)c->u[j] / ((double)c->omega[j] * rhoj);
    double mj = c->mass ? (double)c->mass[j] : c->mass_scalar;
    double sg = k_sigma(p->kernel);
    double Fi = r < Hi ? sg / (Hi * Hi * Hi * Hi) * k_dw(p->kernel, r / Hi) : 0.0;
    double Fj = r < Hj ? sg / (Hj * Hj * Hj * Hj) * k_dw(p->kernel, r / Hj) : 0.0;
    double rh[3] = {d[0] / r, d[1] / r, d[2] / r};
    double vr = 0.0;
    for (int a = 0; a < 3; a++) vr += ((double)c->vel[3 * i + a] - (double)c->vel[3 * j + a]) * rh[a];
    double mu = vr < 0.0 ? vr : 0.0;
    double vs = ci + cj - 3.0 * mu;
    double Pi = -0.5 * p->alpha * vs * mu / (0.5 * (rhoi + rhoj));
    double Fbar = 0.5 * (Fi + Fj);
    double t = mj * (Ai * Fi + Aj * Fj + Pi * Fbar);
    for (int a = 0; a < 3; a++) f->a[a] -= t * rh[a];
    f->asum += fabs(t);
    f->asq += t * t;
    double e = mj * (Ai * Fi + 0.5 * Pi * Fbar) * vr;
    f->du += e;
    f->dusum += fabs(e);
    f->dusq += e * e;
    f->duvisc += mj * 0.5 * Pi * Fbar * vr;
    if (vs > f->vsig) f->vsig = vs;
}

int orc_hydro_force(const orc_params *p, int64_t n, const float *pos, const float *vel, const float *u,
                    const float *mass, double mass_scalar, const float *h, const float *rho, const float *omega,
                    const int32_t *active, int64_t n_active, int brute, double cell_hint,
                    double *acc, double *dudt, double *vsig, double *asum, double *dusum, double *duvisc,
                    int64_t *npair, uint8_t *edge, double *asq, double *dusq)
{
    orc_grid *g = brute ? NULL : grid_build(n, pos, p->box, cell_hint, h);
    force_ctx c = {p, n, pos, vel, u, mass, h, rho, omega, mass_scalar};
    double hglob = 0.0;
    for (int64_t i = 0; i < n; i++)
        if ((double)h[i] > hglob) hglob = (double)h[i];
    int64_t na = active ? n_active : n;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        force_acc f;
        memset(&f, 0, sizeof(f));
        if (!g) {
            for (int64_t j = 0; j < n; j++) force_pair(&c, i, j, &f);
        } else {
            double xi[3] = {(double)pos[3 * i], (double)pos[3 * i + 1], (double)pos[3 * i + 2]};
            double Hi = (double)h[i];
            int lo[3], cnt[3];
            for (int ax = 0; ax < 3; ax++) axis_range(g, xi[ax], hglob * (1.0 + 2e-6), &lo[ax], &cnt[ax]);
            for (int kz = 0; kz < cnt[2]; kz++)
                for (int ky = 0; ky < cnt[1]; ky++)
                    for (int kx = 0; kx < cnt[0]; kx++) {
                        int cx = ((lo[0] + kx) % g->G + g->G) % g->G;
                        int cy = ((lo[1] + ky) % g->G + g->G) % g->G;
                        int cz = ((lo[2] + kz) % g->G + g->G) % g->G;
                        int64_t cc = ((int64_t)cz * g->G + cy) * g->G + cx;
                        if (g->start[cc] == g->start[cc + 1]) continue;
                        double reach = (Hi > g->hmax[cc] ? Hi : g->hmax[cc]) * (1.0 + 2e-6);
                        if (cell_mindist2(g, xi, cx, cy, cz) > reach * reach) continue; /* pruning only */
                        for (int64_t s = g->start[cc]; s < g->start[cc + 1]; s++) force_pair(&c, i, g->idx[s], &f);
                    }
        }
        acc[3 * a] = f.a[0]; acc[3 * a + 1] = f.a[1]; acc[3 * a + 2] = f.a[2];
        dudt[a] = f.du; vsig[a] = f.vsig;
        if (asum) asum[a] = f.asum;
        if (dusum) dusum[a] = f.dusum;
        if (duvisc) duvisc[a] = f.duvisc;
        if (asq) asq[a] = f.asq;
        if (dusq) dusq[a] = f.dusq;
        if (npair) npair[a] = f.npair;
        if (edge) edge[a] = (uint8_t)(f.edge ? ORC_E_RADIUS : 0);
    }
    grid_free(g);
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ================================================================ improved-SPH extension
 * "Improved SPH" of the paper's ref [6] (PAPER.md:25 §1, :209): the paper only cites it.  What is stated
 * here are the READINGS R17-R20 of DESIGN.md, restated from the published lineage (velocity-gradient
 * estimators of the Gadget lineage [2]; shear limiter of Balsara; time-dependent viscosity of Morris &
 * Monaghan; artificial conduction in the signal-velocity form of Price).
 *
 * R17  velocity divergence and curl with the particle's own support radius (gather form, no grad-h factor):
 *        (div v)_i  = (1/rho_i) sum_j m_j (v_j - v_i) . grad_i W_ij(H_i)
 *        (curl v)_i = (1/rho_i) sum_j m_j (v_i - v_j) x grad_i W_ij(H_i),   grad_i W_ij = dW/dr(r_ij, H_i) rhat_ij,
 *      rhat_ij = (x_i - x_j)/r_ij, over j != i with r_ij < H_i.
 * R18  shear limiter  f_i = |div v_i| / (|div v_i| + |curl v_i| + 1e-4 c_i / H_i);  Pi_ij is multiplied by (f_i + f_j)/2.
 * R19  per-particle viscosity coefficient alpha_i (input): Pi_ij uses (alpha_i + alpha_j)/2 in place of alpha;
 *      its evolution equation  d alpha_i/dt = -(alpha_i - alpha_min) / tau_i + S_i,
 *      tau_i = H_i / (2 l c_i),  S_i = max(0, -div v_i) (alpha_max - alpha_i).
 * R20  artificial conduction: du_i/dt += sum_j m_j alpha_c vsig^u_ij (u_i - u_j) Fbar_ij / rhobar_ij,
 *      vsig^u_ij = sqrt(|P_i - P_j| / rhobar_ij), Fbar = (F_ij(H_i) + F_ij(H_j))/2 (<= 0), same pair set as the force.
 * Everything else (pair set, pressure terms, signal velocity, v_sig maximum) is R8-R12 unchanged.
 */
typedef struct {
    double alpha_min, alpha_max, decay_l; /* R19 */
    double alpha_cond;                    /* R20; 0 switches conduction off */
    int balsara;                          /* R18 on/off */
} orc_improved;

int orc_velocity_gradients(const orc_params *p, int64_t n, const float *pos, const float *vel, const float *mass,
                           double mass_scalar, const float *h, const float *rho, const int32_t *active, int64_t n_active,
                           double *divv, double *curlv /* na*3 */)
{
    int64_t na = active ? n_active : n;
    double L = p->box;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        double Hi = (double)h[i], dv = 0.0, cx = 0.0, cy = 0.0, cz = 0.0;
        for (int64_t j = 0; j < n; j++) { /* plain definition: all j (brute force) */
            if (j == i) continue;
            double d[3];
            for (int k = 0; k < 3; k++) d[k] = min_image((double)pos[3 * i + k] - (double)pos[3 * j + k], L);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (!(r2 < Hi * Hi) || r2 == 0.0) continue;
            double r = sqrt(r2);
            double mj = mass ? (double)mass[j] : mass_scalar;
            double g = mj * orc_dWdr(p->kernel, r, Hi) / r; /* m_j dW/dr / r: grad W = g/m_j * d */
            double w[3];
            for (int k = 0; k < 3; k++) w[k] = (double)vel[3 * j + k] - (double)vel[3 * i + k];
            dv += g * (w[0] * d[0] + w[1] * d[1] + w[2] * d[2]);
            cx -= g * (w[1] * d[2] - w[2] * d[1]); /* (v_i - v_j) x grad W = -w x grad W */
            cy -= g * (w[2] * d[0] - w[0] * d[2]);
            cz -= g * (w[0] * d[1] - w[1] * d[0]);
        }
        double ir = 1.0 / (double)rho[i];
        divv[a] = dv * ir;
        curlv[3 * a] = cx * ir; curlv[3 * a + 1] = cy * ir; curlv[3 * a + 2] = cz * ir;
    }
    return 0;
}

/* R18 */
static double balsara_f(double divv, const float *curl, double c, double H)
{
    double cm = sqrt((double)curl[0] * curl[0] + (double)curl[1] * curl[1] + (double)curl[2] * curl[2]);
    return fabs(divv) / (fabs(divv) + cm + 1e-4 * c / H);
}

int orc_hydro_force_improved(const orc_params *p, const orc_improved *q, int64_t n, const float *pos, const float *vel,
                             const float *u, const float *mass, double mass_scalar, const float *h, const float *rho,
                             const float *omega, const float *alpha, const float *divv, const float *curlv,
                             const int32_t *active, int64_t n_active, double *acc, double *dudt, double *vsig,
                             double *dalpha, double *asum, double *dusum, double *asq, double *dusq, double *ducond)
{
    int64_t na = active ? n_active : n;
    double L = p->box, gm1 = p->gamma - 1.0, sg = k_sigma(p->kernel);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        double Hi = (double)h[i], rhoi = (double)rho[i], ui = (double)u[i];
        double ci = sqrt(p->gamma * gm1 * ui), Pi_ = gm1 * rhoi * ui;
        double Ai = gm1 * ui / ((double)omega[i] * rhoi);
        double fi = q->balsara ? balsara_f((double)divv[i], curlv + 3 * i, ci, Hi) : 1.0;
        double ax = 0, ay = 0, az = 0, du = 0, vs = 0, as = 0, dus = 0, a2 = 0, du2 = 0, duc = 0;
        for (int64_t j = 0; j < n; j++) { /* plain definition: all j (brute force) */
            if (j == i) continue;
            double d[3];
            for (int k = 0; k < 3; k++) d[k] = min_image((double)pos[3 * i + k] - (double)pos[3 * j + k], L);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            double Hj = (double)h[j], Hm = Hi > Hj ? Hi : Hj;
            if (!(r2 < Hm * Hm)) continue;
            double uj = (double)u[j], rhoj = (double)rho[j];
            double cj = sqrt(p->gamma * gm1 * uj);
            if (r2 == 0.0) { if (ci + cj > vs) vs = ci + cj; continue; }
            double r = sqrt(r2);
            double Aj = gm1 * uj / ((double)omega[j] * rhoj);
            double mj = mass ? (double)mass[j] : mass_scalar;
            double Fi = r < Hi ? sg / (Hi * Hi * Hi * Hi) * k_dw(p->kernel, r / Hi) : 0.0;
            double Fj = r < Hj ? sg / (Hj * Hj * Hj * Hj) * k_dw(p->kernel, r / Hj) : 0.0;
            double vr = 0.0;
            for (int k = 0; k < 3; k++) vr += ((double)vel[3 * i + k] - (double)vel[3 * j + k]) * d[k] / r;
            double mu = vr < 0.0 ? vr : 0.0;
            double vsij = ci + cj - 3.0 * mu;
            double rb = 0.5 * (rhoi + rhoj);
            double aij = 0.5 * ((double)alpha[i] + (double)alpha[j]);                                       /* R19 */
            double fj = q->balsara ? balsara_f((double)divv[j], curlv + 3 * j, cj, Hj) : 1.0;
            double PI = -0.5 * aij * vsij * mu / rb * 0.5 * (fi + fj);                                       /* R9, R18 */
            double Fbar = 0.5 * (Fi + Fj);
            double t = mj * (Ai * Fi + Aj * Fj + PI * Fbar);
            ax -= t * d[0] / r; ay -= t * d[1] / r; az -= t * d[2] / r;
            as += fabs(t); a2 += t * t;
            double e = mj * (Ai * Fi + 0.5 * PI * Fbar) * vr;
            double Pj_ = gm1 * rhoj * uj;
            double ec = mj * q->alpha_cond * sqrt(fabs(Pi_ - Pj_) / rb) * (ui - uj) * Fbar / rb;             /* R20 */
            du += e + ec; duc += ec;
            dus += fabs(e) + fabs(ec); du2 += e * e + ec * ec;
            if (vsij > vs) vs = vsij;
        }
        acc[3 * a] = ax; acc[3 * a + 1] = ay; acc[3 * a + 2] = az;
        dudt[a] = du; vsig[a] = vs;
        double tau = Hi / (2.0 * q->decay_l * ci);
        double S = ((double)divv[i] < 0.0 ? -(double)divv[i] : 0.0) * (q->alpha_max - (double)alpha[i]);
        dalpha[a] = -((double)alpha[i] - q->alpha_min) / tau + S;                                            /* R19 */
        if (asum) asum[a] = as;
        if (dusum) dusum[a] = dus;
        if (asq) asq[a] = a2;
        if (dusq) dusq[a] = du2;
        if (ducond) ducond[a] = duc;
    }
    return 0;
}

/* ================================================================ thermal conduction
 * The paper ports "thermal conduction" as a third module of the same pattern (PAPER.md:27 §1, :41: ~14 % of the
 * run time, :102 §2.4, :156 §3.3) and gives no equation.  READING R21, the isotropic SPH heat
 * conduction estimate of the published lineage (second-derivative form of Brookshaw with the harmonic mean of the
 * conductivities of Cleary & Monaghan, as used for conduction in the Gadget lineage), over the symmetric pair set
 * r_ij < max(H_i, H_j) of the force pass:
 *   du_i/dt = sum_j m_j / (rho_i rho_j) * [4 kappa_i kappa_j / (kappa_i + kappa_j)] * (T_i - T_j) * Fbar_ij / r_ij,
 *   Fbar_ij = (F_ij(H_i) + F_ij(H_j))/2 <= 0,  T = u (the constants of the temperature scale are absorbed in
 *   kappa_0),  kappa_i = kappa_0 T_i^e  (e = 5/2: Spitzer; e = 0: constant conductivity).
 * Heat flows from hot to cold; the pair term is antisymmetric in i <-> j (energy is conserved pair by pair).
 */
int orc_thermal_conduction(const orc_params *p, int64_t n, const float *pos, const float *u, const float *mass,
                           double mass_scalar, const float *h, const float *rho, double kappa0, double kappa_exp,
                           const int32_t *active, int64_t n_active, double *dudt, double *dusum, double *dusq)
{
    int64_t na = active ? n_active : n;
    double L = p->box, sg = k_sigma(p->kernel);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        double Hi = (double)h[i], Ti = (double)u[i], ki = kappa0 * pow(Ti, kappa_exp);
        double du = 0.0, s1 = 0.0, s2 = 0.0;
        for (int64_t j = 0; j < n; j++) { /* plain definition: all j (brute force) */
            if (j == i) continue;
            double d[3];
            for (int k = 0; k < 3; k++) d[k] = min_image((double)pos[3 * i + k] - (double)pos[3 * j + k], L);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            double Hj = (double)h[j], Hm = Hi > Hj ? Hi : Hj;
            if (!(r2 < Hm * Hm) || r2 == 0.0) continue;
            double r = sqrt(r2);
            double Fi = r < Hi ? sg / (Hi * Hi * Hi * Hi) * k_dw(p->kernel, r / Hi) : 0.0;
            double Fj = r < Hj ? sg / (Hj * Hj * Hj * Hj) * k_dw(p->kernel, r / Hj) : 0.0;
            double Tj = (double)u[j], kj = kappa0 * pow(Tj, kappa_exp);
            double mj = mass ? (double)mass[j] : mass_scalar;
            double kij = (ki + kj) > 0.0 ? 4.0 * ki * kj / (ki + kj) : 0.0;
            double e = mj / ((double)rho[i] * (double)rho[j]) * kij * (Ti - Tj) * 0.5 * (Fi + Fj) / r;
            du += e; s1 += fabs(e); s2 += e * e;
        }
        dudt[a] = du;
        if (dusum) dusum[a] = s1;
        if (dusq) dusq[a] = s2;
    }
    return 0;
}

/* ================================================================ short-range gravity
 * The paper's gravity is "Barnes-Hut + Particle-Mesh" (§1), i.e. a TreePM split: the tree walk
 * computes the SHORT-range part (PAPER.md:41 ~15 % of the time, :102-104 §2.4: "particles interact with distant
 * tree nodes as they were point-like pseudo particles"); no formulas are given.  READING R23, the
 * short-range force of the TreePM split of the Gadget lineage [2], with Plummer softening, minimum image, and an
 * explicit truncation radius (the factor is 2e-3 at 4.5 r_s and the lineage stops the walk there):
 *   a_i = - G sum_{j != i, r_ij < r_cut} m_j d_ij / (r_ij^2 + eps^2)^(3/2) * [erfc(r_ij / 2 r_s) + r_ij / (r_s sqrt(pi)) exp(-r_ij^2 / 4 r_s^2)]
 * This is the exact definition (direct summation).  The tree code on the GPU reaches it up to the multipole
 * error of its opening criterion (exactly, for an opening angle of zero).
 */
int orc_gravity_short(const orc_params *p, int64_t n, const float *pos, const float *mass, double mass_scalar, double G,
                      double r_s, double r_cut, double eps, const int32_t *active, int64_t n_active, double *acc,
                      double *asum)
{
    int64_t na = active ? n_active : n;
    double L = p->box;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t a = 0; a < na; a++) {
        int64_t i = active ? active[a] : a;
        double ax = 0, ay = 0, az = 0, s = 0;
        for (int64_t j = 0; j < n; j++) {
            if (j == i) continue;
            double d[3];
            for (int k = 0; k < 3; k++) d[k] = min_image((double)pos[3 * i + k] - (double)pos[3 * j + k], L);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (!(r2 < r_cut * r_cut)) continue;
            double r = sqrt(r2), x = r / (2.0 * r_s);
            double fac = erfc(x) + r / (r_s * sqrt(M_PI)) * exp(-x * x);
            double mj = mass ? (double)mass[j] : mass_scalar;
            double t = G * mj * fac / ((r2 + eps * eps) * sqrt(r2 + eps * eps));
            ax -= t * d[0]; ay -= t * d[1]; az -= t * d[2];
            s += t * r;
        }
        acc[3 * a] = ax; acc[3 * a + 1] = ay; acc[3 * a + 2] = az;
        if (asum) asum[a] = s;
    }
    return 0;
}
