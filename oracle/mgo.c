/* mgo.c -- CPU oracle (test infrastructure; see mgo.h for scope, citations and pins).
 *
 * Plain triple loops, fp64, one code path for all levels (explicit minus-face arrays
 * on every level).  Expression trees follow SURVEY.md §8(c) C1-C9 / DESIGN.md §3
 * literally; compile with -ffp-contract=off so that only the fma() calls written
 * here are fused.  OpenMP, when enabled, only splits the k loop of loops whose
 * iterations are independent (one colour of a half-sweep, residual, transfers), so
 * every field is bit-identical to the single-thread run; sums are accumulated per
 * k-plane in long double and then added in plane order (thread-count independent).
 */
#include "mgo.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MGO_MAX_LEVELS 32

typedef struct {
    int nx, ny, nz;
    double h, h2, ih2;          /* C1 */
    double *bx, *by, *bz;       /* minus-face coefficients */
    double *wx, *wy, *wz;       /* R24: plus-wall face coefficients of a non-periodic axis:
                                 * wx[j + ny*k] belongs to cell (nx-1, j, k), wy[i + nx*k], wz[i + nx*j] */
    int walled[3];              /* axis is not periodic: walls at both ends (R24) */
    double *p, *f;              /* levels >= 1: correction e and restricted rhs */
    double *r;                  /* residual scratch (levels that have a coarser one) */
} level_t;

struct mgo_solver {
    int nlev;
    int bc[3];                  /* per axis, as given to mgo_create (both sides alike) */
    int bcm[3], bcp[3];         /* R24: per side (minus, plus): MGO_BC_PERIODIC / NEUMANN / DIRICHLET */
    int nu1, nu2, coarse_sweeps;
    int cycle_type;             /* R23: MGO_CYCLE_V / F / W */
    level_t lv[MGO_MAX_LEVELS];
};

static int g_threads = 0; /* 0 = library default */

int mgo_threads(void)
{
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

void mgo_set_threads(int n)
{
    g_threads = n;
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#endif
}

static size_t lv_cells(const level_t *L) { return (size_t)L->nx * L->ny * L->nz; }

#define IDX(L, i, j, k) ((size_t)(i) + (size_t)(L)->nx * ((size_t)(j) + (size_t)(L)->ny * (size_t)(k)))

/* ------------------------------------------------------------------ create */
int mgo_create(int nx, int ny, int nz, double h, const int bc[3], mgo_solver **out)
{
    if (!out || !bc) return MGO_EINVAL;
    *out = NULL;
    for (int a = 0; a < 3; ++a)
        if (bc[a] != 0 && bc[a] != 1) return MGO_EINVAL;
    const int bc6[6] = { bc[0], bc[0], bc[1], bc[1], bc[2], bc[2] };
    return mgo_create6(nx, ny, nz, h, bc6, out);
}

/* R24: one boundary type per side, order x-, x+, y-, y+, z-, z+.  Periodic comes in pairs. */
int mgo_create6(int nx, int ny, int nz, double h, const int bc6[6], mgo_solver **out)
{
    if (!out || !bc6) return MGO_EINVAL;
    *out = NULL;
    if (nx < 4 || ny < 4 || nz < 4 || (nx & 1) || (ny & 1) || (nz & 1)) return MGO_EINVAL;
    if (!(h > 0.0) || !isfinite(h)) return MGO_EINVAL;
    for (int a = 0; a < 3; ++a) {
        const int m = bc6[2 * a], q = bc6[2 * a + 1];
        if (m < MGO_BC_PERIODIC || m > MGO_BC_DIRICHLET || q < MGO_BC_PERIODIC || q > MGO_BC_DIRICHLET) return MGO_EINVAL;
        if ((m == MGO_BC_PERIODIC) != (q == MGO_BC_PERIODIC)) return MGO_EINVAL;
    }

    mgo_solver *s = (mgo_solver *)calloc(1, sizeof(*s));
    if (!s) return MGO_ENOMEM;
    for (int a = 0; a < 3; ++a) {
        s->bcm[a] = bc6[2 * a]; s->bcp[a] = bc6[2 * a + 1];
        s->bc[a] = s->bcm[a] == MGO_BC_PERIODIC ? 0 : 1;
    }
    s->nu1 = 2; s->nu2 = 2; s->coarse_sweeps = 32;

    /* R7: halve every axis while the halved dims stay even (so red-black colouring is
     * consistent across a periodic wrap on every level) and the smallest dim is > 4. */
    int n[3] = { nx, ny, nz };
    double hl = h;
    int l = 0;
    for (;;) {
        level_t *L = &s->lv[l];
        L->nx = n[0]; L->ny = n[1]; L->nz = n[2];
        L->h = hl; L->h2 = hl * hl; L->ih2 = 1.0 / L->h2;
        for (int a = 0; a < 3; ++a) L->walled[a] = s->bcm[a] != MGO_BC_PERIODIC;
        ++l;
        int mn = n[0] < n[1] ? n[0] : n[1]; if (n[2] < mn) mn = n[2];
        if (mn <= 4 || (n[0] % 4) || (n[1] % 4) || (n[2] % 4) || l == MGO_MAX_LEVELS) break;
        n[0] /= 2; n[1] /= 2; n[2] /= 2; hl *= 2.0;
    }
    s->nlev = l;
    for (l = 0; l < s->nlev; ++l) {
        level_t *L = &s->lv[l];
        size_t N = lv_cells(L);
        L->bx = (double *)malloc(N * sizeof(double));
        L->by = (double *)malloc(N * sizeof(double));
        L->bz = (double *)malloc(N * sizeof(double));
        L->wx = (double *)calloc((size_t)L->ny * L->nz, sizeof(double));
        L->wy = (double *)calloc((size_t)L->nx * L->nz, sizeof(double));
        L->wz = (double *)calloc((size_t)L->nx * L->ny, sizeof(double));
        if (l > 0) {
            L->p = (double *)malloc(N * sizeof(double));
            L->f = (double *)malloc(N * sizeof(double));
        }
        if (l < s->nlev - 1) L->r = (double *)malloc(N * sizeof(double));
        if (!L->bx || !L->by || !L->bz || !L->wx || !L->wy || !L->wz || (l > 0 && (!L->p || !L->f)) ||
            (l < s->nlev - 1 && !L->r)) { mgo_destroy(s); return MGO_ENOMEM; }
    }
    /* default density rho == 1 */
    {
        level_t *L = &s->lv[0];
        size_t N = lv_cells(L);
        double *one = (double *)malloc(N * sizeof(double));
        if (!one) { mgo_destroy(s); return MGO_ENOMEM; }
        for (size_t c = 0; c < N; ++c) one[c] = 1.0;
        mgo_set_density(s, one);
        free(one);
    }
    *out = s;
    return MGO_OK;
}

void mgo_destroy(mgo_solver *s)
{
    if (!s) return;
    for (int l = 0; l < s->nlev; ++l) {
        free(s->lv[l].bx); free(s->lv[l].by); free(s->lv[l].bz);
        free(s->lv[l].wx); free(s->lv[l].wy); free(s->lv[l].wz);
        free(s->lv[l].p); free(s->lv[l].f); free(s->lv[l].r);
    }
    free(s);
}

int mgo_set_cycle(mgo_solver *s, int nu1, int nu2, int coarse_sweeps)
{
    if (!s || nu1 < 0 || nu2 < 0 || coarse_sweeps < 1) return MGO_EINVAL;
    s->nu1 = nu1; s->nu2 = nu2; s->coarse_sweeps = coarse_sweeps;
    return MGO_OK;
}

/* ------------------------------------------------------------ coefficients */
int mgo_set_density(mgo_solver *s, const double *rho)
{
    if (!s || !rho) return MGO_EINVAL;
    level_t *L = &s->lv[0];
    const int nx = L->nx, ny = L->ny, nz = L->nz;
    size_t N = lv_cells(L);
    for (size_t c = 0; c < N; ++c)
        if (!(rho[c] > 0.0) || !isfinite(rho[c])) return MGO_EINVAL;

    /* C2: a = 0.5/rho per cell; face between cells c and nb: beta = a[c] + a[nb];
     * Neumann wall face: beta = +0.0.  (R4: beta = 1/rho_face, rho_face harmonic mean)
     * R24 / C2w: Dirichlet wall face (p = 0 ON the face, ghost = -p_c, ghost density = the cell's):
     * beta_w (0 - p_c) with beta_w = 2.0 * (a[c] + a[c]). */
    double *a = (double *)malloc(N * sizeof(double));
    if (!a) return MGO_ENOMEM;
    for (size_t c = 0; c < N; ++c) a[c] = 0.5 / rho[c];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t c = IDX(L, i, j, k);
                int im = i == 0 ? nx - 1 : i - 1;
                int jm = j == 0 ? ny - 1 : j - 1;
                int km = k == 0 ? nz - 1 : k - 1;
                const double wall = 2.0 * (a[c] + a[c]);
                L->bx[c] = (i == 0 && s->bcm[0] != MGO_BC_PERIODIC) ? (s->bcm[0] == MGO_BC_DIRICHLET ? wall : 0.0)
                                                                    : a[c] + a[IDX(L, im, j, k)];
                L->by[c] = (j == 0 && s->bcm[1] != MGO_BC_PERIODIC) ? (s->bcm[1] == MGO_BC_DIRICHLET ? wall : 0.0)
                                                                    : a[c] + a[IDX(L, i, jm, k)];
                L->bz[c] = (k == 0 && s->bcm[2] != MGO_BC_PERIODIC) ? (s->bcm[2] == MGO_BC_DIRICHLET ? wall : 0.0)
                                                                    : a[c] + a[IDX(L, i, j, km)];
                if (i == nx - 1) L->wx[j + (size_t)ny * k] = s->bcp[0] == MGO_BC_DIRICHLET ? wall : 0.0;
                if (j == ny - 1) L->wy[i + (size_t)nx * k] = s->bcp[1] == MGO_BC_DIRICHLET ? wall : 0.0;
                if (k == nz - 1) L->wz[i + (size_t)nx * j] = s->bcp[2] == MGO_BC_DIRICHLET ? wall : 0.0;
            }
    free(a);

    /* C3 (R8): coarse face = arithmetic mean of the 4 finer faces lying on it */
    for (int l = 1; l < s->nlev; ++l) {
        const level_t *F = &s->lv[l - 1];
        level_t *C = &s->lv[l];
#pragma omp parallel for schedule(static)
        for (int K = 0; K < C->nz; ++K)
            for (int J = 0; J < C->ny; ++J)
                for (int I = 0; I < C->nx; ++I) {
                    const int i = 2 * I, j = 2 * J, k = 2 * K;
                    size_t c = IDX(C, I, J, K);
                    C->bx[c] = 0.25 * ((F->bx[IDX(F, i, j, k)] + F->bx[IDX(F, i, j + 1, k)]) +
                                       (F->bx[IDX(F, i, j, k + 1)] + F->bx[IDX(F, i, j + 1, k + 1)]));
                    C->by[c] = 0.25 * ((F->by[IDX(F, i, j, k)] + F->by[IDX(F, i + 1, j, k)]) +
                                       (F->by[IDX(F, i, j, k + 1)] + F->by[IDX(F, i + 1, j, k + 1)]));
                    C->bz[c] = 0.25 * ((F->bz[IDX(F, i, j, k)] + F->bz[IDX(F, i + 1, j, k)]) +
                                       (F->bz[IDX(F, i, j + 1, k)] + F->bz[IDX(F, i + 1, j + 1, k)]));
                }
        /* the plus walls coarsen by the same rule (the four finer wall faces on the coarse one) */
        for (int K = 0; K < C->nz; ++K)
            for (int J = 0; J < C->ny; ++J) {
                const size_t m = F->ny;
                C->wx[J + (size_t)C->ny * K] = 0.25 * ((F->wx[2 * J + m * (2 * K)] + F->wx[2 * J + 1 + m * (2 * K)]) +
                                                       (F->wx[2 * J + m * (2 * K + 1)] + F->wx[2 * J + 1 + m * (2 * K + 1)]));
            }
        for (int K = 0; K < C->nz; ++K)
            for (int I = 0; I < C->nx; ++I) {
                const size_t m = F->nx;
                C->wy[I + (size_t)C->nx * K] = 0.25 * ((F->wy[2 * I + m * (2 * K)] + F->wy[2 * I + 1 + m * (2 * K)]) +
                                                       (F->wy[2 * I + m * (2 * K + 1)] + F->wy[2 * I + 1 + m * (2 * K + 1)]));
            }
        for (int J = 0; J < C->ny; ++J)
            for (int I = 0; I < C->nx; ++I) {
                const size_t m = F->nx;
                C->wz[I + (size_t)C->nx * J] = 0.25 * ((F->wz[2 * I + m * (2 * J)] + F->wz[2 * I + 1 + m * (2 * J)]) +
                                                       (F->wz[2 * I + m * (2 * J + 1)] + F->wz[2 * I + 1 + m * (2 * J + 1)]));
            }
    }
    return MGO_OK;
}

/* ------------------------------------------------------------- the stencil */
/* C4: neighbour sum S and diagonal D of cell (i,j,k), order x-,x+,y-,y+,z-,z+.
 * At a wall (non-periodic axis, R5 / R24) the face coefficient is the stored wall value (minus
 * wall: entry 0 of the minus-face array; plus wall: wx / wy / wz) and the neighbour value is 0.0
 * (C2: Neumann wall 0.0 * 0.0; Dirichlet wall beta_w * 0.0 with beta_w in D). */
static inline void stencil(const level_t *L, const double *p, int i, int j, int k,
                           double *S, double *D)
{
    const int nx = L->nx, ny = L->ny, nz = L->nz;
    const int im = i == 0 ? nx - 1 : i - 1, ip = i == nx - 1 ? 0 : i + 1;
    const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
    const int km = k == 0 ? nz - 1 : k - 1, kp = k == nz - 1 ? 0 : k + 1;
    const int wxm = L->walled[0] && i == 0, wxp = L->walled[0] && i == nx - 1;
    const int wym = L->walled[1] && j == 0, wyp = L->walled[1] && j == ny - 1;
    const int wzm = L->walled[2] && k == 0, wzp = L->walled[2] && k == nz - 1;
    const double bxm = L->bx[IDX(L, i, j, k)], bxp = wxp ? L->wx[j + (size_t)ny * k] : L->bx[IDX(L, ip, j, k)];
    const double bym = L->by[IDX(L, i, j, k)], byp = wyp ? L->wy[i + (size_t)nx * k] : L->by[IDX(L, i, jp, k)];
    const double bzm = L->bz[IDX(L, i, j, k)], bzp = wzp ? L->wz[i + (size_t)nx * j] : L->bz[IDX(L, i, j, kp)];
    const double pxm = wxm ? 0.0 : p[IDX(L, im, j, k)], pxp = wxp ? 0.0 : p[IDX(L, ip, j, k)];
    const double pym = wym ? 0.0 : p[IDX(L, i, jm, k)], pyp = wyp ? 0.0 : p[IDX(L, i, jp, k)];
    const double pzm = wzm ? 0.0 : p[IDX(L, i, j, km)], pzp = wzp ? 0.0 : p[IDX(L, i, j, kp)];
    *S = fma(bzp, pzp, fma(bzm, pzm, fma(byp, pyp, fma(bym, pym, fma(bxp, pxp, bxm * pxm)))));
    *D = ((((bxm + bxp) + bym) + byp) + bzm) + bzp;
}

static void smooth_half(const level_t *L, int colour, const double *f, double *p)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L->nz; ++k)
        for (int j = 0; j < L->ny; ++j)
            for (int i = (j + k + colour) & 1; i < L->nx; i += 2) {
                double S, D;
                stencil(L, p, i, j, k, &S, &D);
                const double invD = 1.0 / D;                       /* C5 */
                p[IDX(L, i, j, k)] = fma(-L->h2, f[IDX(L, i, j, k)], S) * invD;
            }
}

/* R9: one sweep = red (colour 0) half-sweep, then black (colour 1) */
static void sweep(const level_t *L, const double *f, double *p)
{
    smooth_half(L, 0, f, p);
    smooth_half(L, 1, f, p);
}

static void residual(const level_t *L, const double *f, const double *p, double *r)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L->nz; ++k)
        for (int j = 0; j < L->ny; ++j)
            for (int i = 0; i < L->nx; ++i) {
                double S, D;
                stencil(L, p, i, j, k, &S, &D);
                size_t c = IDX(L, i, j, k);
                r[c] = fma(-L->ih2, fma(-D, p[c], S), f[c]);       /* C6 */
            }
}

static void apply(const level_t *L, const double *p, double *out)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L->nz; ++k)
        for (int j = 0; j < L->ny; ++j)
            for (int i = 0; i < L->nx; ++i) {
                double S, D;
                stencil(L, p, i, j, k, &S, &D);
                size_t c = IDX(L, i, j, k);
                out[c] = L->ih2 * fma(-D, p[c], S);
            }
}

/* C7 (R11): coarse rhs = mean of the 8 children */
static void restrict8(const level_t *F, const level_t *C, const double *r, double *fc)
{
#pragma omp parallel for schedule(static)
    for (int K = 0; K < C->nz; ++K)
        for (int J = 0; J < C->ny; ++J)
            for (int I = 0; I < C->nx; ++I) {
                const int i = 2 * I, j = 2 * J, k = 2 * K;
                const double r000 = r[IDX(F, i, j, k)],         r100 = r[IDX(F, i + 1, j, k)];
                const double r010 = r[IDX(F, i, j + 1, k)],     r110 = r[IDX(F, i + 1, j + 1, k)];
                const double r001 = r[IDX(F, i, j, k + 1)],     r101 = r[IDX(F, i + 1, j, k + 1)];
                const double r011 = r[IDX(F, i, j + 1, k + 1)], r111 = r[IDX(F, i + 1, j + 1, k + 1)];
                fc[IDX(C, I, J, K)] =
                    0.125 * (((r000 + r100) + (r010 + r110)) + ((r001 + r101) + (r011 + r111)));
            }
}

static inline double lerp(double near, double far) { return fma(0.25, far, 0.75 * near); }

/* neighbour coarse index on the side the fine child leans to: wrap (periodic), the boundary cell
 * itself beyond a wall.  *sign = -1.0 beyond a Dirichlet wall (R24: ghost = -e_boundary, so that
 * the interpolant vanishes on the wall), +1.0 otherwise (Neumann: ghost = e_boundary, R12). */
static inline int far_index(int I, int side, int n, int bc_minus, int bc_plus, double *sign)
{
    int Ip = I + 2 * side - 1;
    *sign = 1.0;
    if (Ip < 0) {
        if (bc_minus == MGO_BC_PERIODIC) Ip = n - 1;
        else { Ip = 0; if (bc_minus == MGO_BC_DIRICHLET) *sign = -1.0; }
    }
    if (Ip >= n) {
        if (bc_plus == MGO_BC_PERIODIC) Ip = 0;
        else { Ip = n - 1; if (bc_plus == MGO_BC_DIRICHLET) *sign = -1.0; }
    }
    return Ip;
}

/* C8 (R12): p += cell-centred trilinear interpolation of e (x first, then y, then z); a value
 * taken beyond Dirichlet walls carries the product of the signs of those axes */
static void prolong_add(const mgo_solver *s, const level_t *F, const level_t *C,
                        const double *e, double *p)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k < F->nz; ++k)
        for (int j = 0; j < F->ny; ++j)
            for (int i = 0; i < F->nx; ++i) {
                const int I = i >> 1, J = j >> 1, K = k >> 1;
                double sx, sy, sz;
                const int Ip = far_index(I, i & 1, C->nx, s->bcm[0], s->bcp[0], &sx);
                const int Jp = far_index(J, j & 1, C->ny, s->bcm[1], s->bcp[1], &sy);
                const int Kp = far_index(K, k & 1, C->nz, s->bcm[2], s->bcp[2], &sz);
                const double v =
                    lerp(lerp(lerp(e[IDX(C, I, J, K)],             sx * e[IDX(C, Ip, J, K)]),
                              lerp(sy * e[IDX(C, I, Jp, K)],       (sx * sy) * e[IDX(C, Ip, Jp, K)])),
                         lerp(lerp(sz * e[IDX(C, I, J, Kp)],       (sx * sz) * e[IDX(C, Ip, J, Kp)]),
                              lerp((sy * sz) * e[IDX(C, I, Jp, Kp)], ((sx * sy) * sz) * e[IDX(C, Ip, Jp, Kp)])));
                p[IDX(F, i, j, k)] = p[IDX(F, i, j, k)] + v;
            }
}

/* C9: plane-ordered long-double sums */
static long double sum_planes(const level_t *L, const double *x, int squared)
{
    long double *part = (long double *)malloc((size_t)L->nz * sizeof(long double));
    size_t plane = (size_t)L->nx * L->ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L->nz; ++k) {
        long double acc = 0.0L;
        const double *q = x + plane * (size_t)k;
        for (size_t c = 0; c < plane; ++c)
            acc += squared ? (long double)q[c] * (long double)q[c] : (long double)q[c];
        part[k] = acc;
    }
    long double tot = 0.0L;
    for (int k = 0; k < L->nz; ++k) tot += part[k];
    free(part);
    return tot;
}

/* R6 / R24: the operator is singular (null space = constants) unless some side is a Dirichlet wall */
static int has_dirichlet(const mgo_solver *s)
{
    for (int a = 0; a < 3; ++a)
        if (s->bcm[a] == MGO_BC_DIRICHLET || s->bcp[a] == MGO_BC_DIRICHLET) return 1;
    return 0;
}

/* ------------------------------------------------------------------ cycle */
/* One multigrid cycle on level l (SURVEY 8(c) "Oracle algorithm"; cycle index per Brandt /
 * Trottenberg et al., DESIGN R23).  type V: the coarse problem is visited once.  type W: twice,
 * the second visit starting from the correction the first one left.  type F: an F-cycle visit
 * followed by a V-cycle visit.  The coarsest level is a fixed number of sweeps (R13) and is
 * visited once per visit of the level above it. */
static void cycle(mgo_solver *s, int l, double *p, const double *f, int type)
{
    level_t *L = &s->lv[l];
    if (l == s->nlev - 1) {                                  /* R13 */
        for (int it = 0; it < s->coarse_sweeps; ++it) sweep(L, f, p);
        return;
    }
    level_t *C = &s->lv[l + 1];
    for (int it = 0; it < s->nu1; ++it) sweep(L, f, p);
    residual(L, f, p, L->r);
    restrict8(L, C, L->r, C->f);
    memset(C->p, 0, lv_cells(C) * sizeof(double));
    cycle(s, l + 1, C->p, C->f, type);
    if (l + 1 < s->nlev - 1) {
        if (type == MGO_CYCLE_W) cycle(s, l + 1, C->p, C->f, MGO_CYCLE_W);
        if (type == MGO_CYCLE_F) cycle(s, l + 1, C->p, C->f, MGO_CYCLE_V);
    }
    prolong_add(s, L, C, C->p, p);
    for (int it = 0; it < s->nu2; ++it) sweep(L, f, p);
}

static void vcycle(mgo_solver *s, int l, double *p, const double *f)
{
    cycle(s, l, p, f, s->cycle_type);
}

int mgo_set_cycle_type(mgo_solver *s, int type)
{
    if (!s || type < MGO_CYCLE_V || type > MGO_CYCLE_W) return MGO_EINVAL;
    s->cycle_type = type;
    return MGO_OK;
}

int mgo_vcycle(mgo_solver *s, const double *rhs, double *p)
{
    if (!s || !rhs || !p) return MGO_EINVAL;
    vcycle(s, 0, p, rhs);
    return MGO_OK;
}

static double residual_norm(mgo_solver *s, const double *rhs, const double *p, double *r_out)
{
    level_t *L = &s->lv[0];
    double *r = r_out ? r_out : (double *)malloc(lv_cells(L) * sizeof(double));
    residual(L, rhs, p, r);
    double nrm = (double)sqrtl(sum_planes(L, r, 1));          /* R15 */
    if (!r_out) free(r);
    return nrm;
}

int mgo_residual(mgo_solver *s, const double *rhs, const double *p, double *r_or_null,
                 double *norm2)
{
    if (!s || !rhs || !p) return MGO_EINVAL;
    double nrm = residual_norm(s, rhs, p, r_or_null);
    if (norm2) *norm2 = nrm;
    return MGO_OK;
}

int mgo_solve(mgo_solver *s, const double *rhs, double *p, double rtol, int max_cycles,
              int *cycles_out, double *relres_out, double *hist)
{
    if (!s || !rhs || !p || !(rtol >= 0.0) || max_cycles < 0) return MGO_EINVAL;
    level_t *L = &s->lv[0];
    const size_t N = lv_cells(L);
    /* R6: singular system (all axes periodic/Neumann): the rhs must be mean-free */
    const int singular = !has_dirichlet(s);
    if (singular) {
        long double mean = sum_planes(L, rhs, 0) / (long double)N;
        long double nrm = sqrtl(sum_planes(L, rhs, 1));
        if (fabsl(mean) > 1e-12L * (nrm / sqrtl((long double)N))) return MGO_EINCOMPATIBLE;
    }
    double r0 = residual_norm(s, rhs, p, NULL);
    if (hist) hist[0] = r0;
    if (!isfinite(r0)) return MGO_EDIVERGED;
    int k = 0, status = MGO_NOT_CONVERGED;
    double rk = r0;
    if (r0 <= rtol * r0) status = MGO_OK;                     /* r0 == 0 */
    while (status != MGO_OK && k < max_cycles) {
        vcycle(s, 0, p, rhs);
        ++k;
        rk = residual_norm(s, rhs, p, NULL);
        if (hist) hist[k] = rk;
        if (!isfinite(rk)) { if (cycles_out) *cycles_out = k; return MGO_EDIVERGED; }
        if (rk <= rtol * r0) status = MGO_OK;
    }
    /* zero arithmetic mean, once, at the end (R6); with a Dirichlet wall p is unique as it is */
    if (singular) {
        double mean = (double)(sum_planes(L, p, 0) / (long double)N);
        for (size_t c = 0; c < N; ++c) p[c] = p[c] - mean;
    }
    if (cycles_out) *cycles_out = k;
    if (relres_out) *relres_out = r0 > 0.0 ? rk / r0 : 0.0;
    return status;
}

/* ----------------------------------------- MG-preconditioned CG (S8(f) rank 1) */
/* R22.  The V-cycle of mgo_vcycle is not a symmetric operator: its post-smoothing repeats the
 * red->black order and its restriction (8-child mean, R11) is not a multiple of the transpose
 * of its prolongation (trilinear, R12).  The preconditioner M of the CG solver is the
 * SYMMETRIC cycle: nu1 red->black sweeps, residual, restriction R' = (1/8) P^T (the transpose
 * of the trilinear prolongation, i.e. the other "full-weighting" reading of R11), coarse
 * correction from zero, prolongation P, nu2 = nu1 black->red sweeps; coarsest level:
 * coarse_sweeps red->black then coarse_sweeps black->red sweeps.  z = M r starts from z = 0.
 *   C14  R'  per axis, x then y then z:  t = w0*r0; t = fma(w1,r1,t); t = fma(w2,r2,t);
 *        t = fma(w3,r3,t) over the fine indices 2I-1, 2I, 2I+1, 2I+2 (wrapped; absent beyond a
 *        Neumann wall: weight 0), w_q = 0.75 [near(i_q) = I] + 0.25 [far(i_q) = I] with near,
 *        far as in C8; finally fc = 0.125 * t.
 *   C12  A d = ih2 * fma(-D, d, S)
 *   C13  PCG (A, M negative definite on the zero-mean subspace; the formulas need no sign):
 *        r = f - A p ; z = M r ; d = z ; rz = r.z ; then per iteration
 *        q = A d ; alpha = rz / (d.q) ; p = fma(alpha,d,p) ; r = fma(-alpha,q,r) ;
 *        stop when ||r|| <= rtol ||r_0|| (r from the recurrence) ;
 *        z = M r ; rz' = r.z ; beta = rz'/rz ; d = fma(beta,d,z).
 *        dot products as C9 (any order, accurate to ~1e-15); mean of p removed at the end. */
static void sweep_rev(const level_t *L, const double *f, double *p)
{
    smooth_half(L, 1, f, p);
    smooth_half(L, 0, f, p);
}

/* weight of coarse index I in the prolongation row of fine index i (C8's near / far rule) */
static inline double pt_weight(int i, int I, int cn, int neumann)
{
    const int near = i >> 1;
    double sign;            /* (periodic or Neumann sides only here: the sign is always +1) */
    const int far = far_index(near, i & 1, cn, neumann, neumann, &sign);
    return (near == I ? 0.75 : 0.0) + (far == I ? 0.25 : 0.0);
}

/* the four fine indices 2I-1 .. 2I+2 that can carry coarse index I, wrapped or (Neumann)
 * clamped with weight 0 when they fall outside */
static inline void pt_stencil(int I, int fn, int cn, int neumann, int idx[4], double w[4])
{
    for (int q = 0; q < 4; ++q) {
        int i = 2 * I - 1 + q;
        int outside = 0;
        if (i < 0) { if (neumann) { outside = 1; i = 0; } else i += fn; }
        if (i >= fn) { if (neumann) { outside = 1; i = fn - 1; } else i -= fn; }
        idx[q] = i;
        w[q] = outside ? 0.0 : pt_weight(i, I, cn, neumann);
    }
}

static void restrict_adj(const mgo_solver *s, const level_t *F, const level_t *C, const double *r, double *fc)
{
#pragma omp parallel for schedule(static)
    for (int K = 0; K < C->nz; ++K)
        for (int J = 0; J < C->ny; ++J)
            for (int I = 0; I < C->nx; ++I) {
                int ix[4], iy[4], iz[4];
                double wx[4], wy[4], wz[4];
                pt_stencil(I, F->nx, C->nx, s->bc[0] == 1, ix, wx);
                pt_stencil(J, F->ny, C->ny, s->bc[1] == 1, iy, wy);
                pt_stencil(K, F->nz, C->nz, s->bc[2] == 1, iz, wz);
                double tz = 0.0;
                for (int c = 0; c < 4; ++c) {
                    double ty = 0.0;
                    for (int b = 0; b < 4; ++b) {
                        double tx = wx[0] * r[IDX(F, ix[0], iy[b], iz[c])];
                        tx = fma(wx[1], r[IDX(F, ix[1], iy[b], iz[c])], tx);
                        tx = fma(wx[2], r[IDX(F, ix[2], iy[b], iz[c])], tx);
                        tx = fma(wx[3], r[IDX(F, ix[3], iy[b], iz[c])], tx);
                        ty = b == 0 ? wy[0] * tx : fma(wy[b], tx, ty);
                    }
                    tz = c == 0 ? wz[0] * ty : fma(wz[c], ty, tz);
                }
                fc[IDX(C, I, J, K)] = 0.125 * tz;
            }
}

static void vcycle_sym(mgo_solver *s, int l, double *p, const double *f)
{
    level_t *L = &s->lv[l];
    if (l == s->nlev - 1) {
        for (int it = 0; it < s->coarse_sweeps; ++it) sweep(L, f, p);
        for (int it = 0; it < s->coarse_sweeps; ++it) sweep_rev(L, f, p);
        return;
    }
    level_t *C = &s->lv[l + 1];
    for (int it = 0; it < s->nu1; ++it) sweep(L, f, p);
    residual(L, f, p, L->r);
    restrict_adj(s, L, C, L->r, C->f);
    memset(C->p, 0, lv_cells(C) * sizeof(double));
    vcycle_sym(s, l + 1, C->p, C->f);
    prolong_add(s, L, C, C->p, p);
    for (int it = 0; it < s->nu2; ++it) sweep_rev(L, f, p);
}

int mgo_restrict_adj(const mgo_solver *s, int level, const double *r, double *fc)
{
    if (!s || level < 0 || level >= s->nlev - 1 || !r || !fc || has_dirichlet(s)) return MGO_EINVAL;
    restrict_adj(s, &s->lv[level], &s->lv[level + 1], r, fc);
    return MGO_OK;
}

/* z = M r: one symmetric cycle from z = 0 */
int mgo_precondition(mgo_solver *s, const double *r, double *z)
{
    if (!s || !r || !z || s->nu1 != s->nu2 || has_dirichlet(s)) return MGO_EINVAL;
    memset(z, 0, lv_cells(&s->lv[0]) * sizeof(double));
    vcycle_sym(s, 0, z, r);
    return MGO_OK;
}

static long double dot_planes(const level_t *L, const double *x, const double *y)
{
    long double *part = (long double *)malloc((size_t)L->nz * sizeof(long double));
    size_t plane = (size_t)L->nx * L->ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L->nz; ++k) {
        long double acc = 0.0L;
        const double *a = x + plane * (size_t)k, *b = y + plane * (size_t)k;
        for (size_t c = 0; c < plane; ++c) acc += (long double)a[c] * (long double)b[c];
        part[k] = acc;
    }
    long double tot = 0.0L;
    for (int k = 0; k < L->nz; ++k) tot += part[k];
    free(part);
    return tot;
}

int mgo_solve_pcg(mgo_solver *s, const double *rhs, double *p, double rtol, int max_iter,
                  int *iters_out, double *relres_out, double *hist)
{
    if (!s || !rhs || !p || !(rtol >= 0.0) || max_iter < 0 || s->nu1 != s->nu2 || has_dirichlet(s)) return MGO_EINVAL;
    level_t *L = &s->lv[0];
    const size_t N = lv_cells(L);
    {
        long double mean = sum_planes(L, rhs, 0) / (long double)N;
        long double nrm = sqrtl(sum_planes(L, rhs, 1));
        if (fabsl(mean) > 1e-12L * (nrm / sqrtl((long double)N))) return MGO_EINCOMPATIBLE;
    }
    double *r = (double *)malloc(N * sizeof(double)), *z = (double *)malloc(N * sizeof(double));
    double *d = (double *)malloc(N * sizeof(double)), *q = (double *)malloc(N * sizeof(double));
    if (!r || !z || !d || !q) { free(r); free(z); free(d); free(q); return MGO_ENOMEM; }
    residual(L, rhs, p, r);
    const double r0 = (double)sqrtl(sum_planes(L, r, 1));
    if (hist) hist[0] = r0;
    int k = 0, status = MGO_NOT_CONVERGED;
    double rk = r0;
    if (!isfinite(r0)) status = MGO_EDIVERGED;
    else if (r0 <= rtol * r0) status = MGO_OK;
    double rz = 0.0;
    if (status == MGO_NOT_CONVERGED && max_iter > 0) {
        memset(z, 0, N * sizeof(double));
        vcycle_sym(s, 0, z, r);
        memcpy(d, z, N * sizeof(double));
        rz = (double)dot_planes(L, r, z);
    }
    while (status == MGO_NOT_CONVERGED && k < max_iter) {
        apply(L, d, q);
        const double dq = (double)dot_planes(L, d, q);
        const double alpha = rz / dq;
#pragma omp parallel for schedule(static)
        for (size_t c = 0; c < N; ++c) {
            p[c] = fma(alpha, d[c], p[c]);
            r[c] = fma(-alpha, q[c], r[c]);
        }
        ++k;
        rk = (double)sqrtl(sum_planes(L, r, 1));
        if (hist) hist[k] = rk;
        if (!isfinite(rk)) { status = MGO_EDIVERGED; break; }
        if (rk <= rtol * r0) { status = MGO_OK; break; }
        if (k == max_iter) break;
        memset(z, 0, N * sizeof(double));
        vcycle_sym(s, 0, z, r);
        const double rz_new = (double)dot_planes(L, r, z);
        const double beta = rz_new / rz;
        rz = rz_new;
#pragma omp parallel for schedule(static)
        for (size_t c = 0; c < N; ++c) d[c] = fma(beta, d[c], z[c]);
    }
    free(r); free(z); free(d); free(q);
    if (status == MGO_EDIVERGED) { if (iters_out) *iters_out = k; return status; }
    {
        double mean = (double)(sum_planes(L, p, 0) / (long double)N);
        for (size_t c = 0; c < N; ++c) p[c] = p[c] - mean;
    }
    if (iters_out) *iters_out = k;
    if (relres_out) *relres_out = r0 > 0.0 ? rk / r0 : 0.0;
    return status;
}

/* ------------------------------------------------- projection steps (S8(f) rank 2) */
/* The two steps either side of the pressure solve in the projection method implied by
 * P:33-36 (eq. 1-2) and stated in BJ:north_star: the right-hand side div(u*)/dt from the
 * staggered intermediate velocity, and the correction u = u* - dt * beta_face * grad p.
 * Staggering (R21): u[i,j,k] lives on the MINUS x-face of cell (i,j,k) (the face bx[i,j,k]
 * belongs to), v on the minus y-face, w on the minus z-face; the plus face of a cell is the
 * next cell's minus face (wrap).  On a Neumann axis the wrap face is the wall (both walls
 * share the entry) and the caller supplies u = 0 there; its beta is 0, so the correction
 * never changes it.
 *   C10  s = 1.0/(h*dt);  f = (((u[i+1]-u[i]) + (v[j+1]-v[j])) + (w[k+1]-w[k])) * s
 *   C11  g = dt/h;        u[i] = fma(-g, bx[i]*(p[i]-p[i-1]), u[i])   (v, w alike)
 * Then div(u_new)/dt = f - A p cell by cell (pinned), i.e. the projected field is
 * divergence-free to the residual of the solve. */
int mgo_project_rhs(const mgo_solver *s, const double *u, const double *v, const double *w,
                    double dt, double *f)
{
    if (!s || !u || !v || !w || !f || !(dt > 0.0) || !isfinite(dt) || has_dirichlet(s)) return MGO_EINVAL;
    const level_t *L = &s->lv[0];
    const int nx = L->nx, ny = L->ny, nz = L->nz;
    const double hd = L->h * dt;
    const double sc = 1.0 / hd;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const int ip = i == nx - 1 ? 0 : i + 1;
                const int jp = j == ny - 1 ? 0 : j + 1;
                const int kp = k == nz - 1 ? 0 : k + 1;
                const size_t c = IDX(L, i, j, k);
                const double du = u[IDX(L, ip, j, k)] - u[c];
                const double dv = v[IDX(L, i, jp, k)] - v[c];
                const double dw = w[IDX(L, i, j, kp)] - w[c];
                f[c] = ((du + dv) + dw) * sc;
            }
    return MGO_OK;
}

int mgo_project_correct(const mgo_solver *s, const double *p, double dt, double *u, double *v, double *w)
{
    if (!s || !u || !v || !w || !p || !(dt > 0.0) || !isfinite(dt) || has_dirichlet(s)) return MGO_EINVAL;
    const level_t *L = &s->lv[0];
    const int nx = L->nx, ny = L->ny, nz = L->nz;
    const double g = dt / L->h;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const int im = i == 0 ? nx - 1 : i - 1;
                const int jm = j == 0 ? ny - 1 : j - 1;
                const int km = k == 0 ? nz - 1 : k - 1;
                const size_t c = IDX(L, i, j, k);
                const double pc = p[c];
                u[c] = fma(-g, L->bx[c] * (pc - p[IDX(L, im, j, k)]), u[c]);
                v[c] = fma(-g, L->by[c] * (pc - p[IDX(L, i, jm, k)]), v[c]);
                w[c] = fma(-g, L->bz[c] * (pc - p[IDX(L, i, j, km)]), w[c]);
            }
    return MGO_OK;
}

/* ------------------------------------------------------- step-level access */
int mgo_num_levels(const mgo_solver *s) { return s ? s->nlev : MGO_EINVAL; }

int mgo_level_dims(const mgo_solver *s, int level, int dims[3], double *h_level)
{
    if (!s || level < 0 || level >= s->nlev) return MGO_EINVAL;
    if (dims) { dims[0] = s->lv[level].nx; dims[1] = s->lv[level].ny; dims[2] = s->lv[level].nz; }
    if (h_level) *h_level = s->lv[level].h;
    return MGO_OK;
}

int mgo_get_walls(const mgo_solver *s, int level, double *wx, double *wy, double *wz)
{
    if (!s || level < 0 || level >= s->nlev) return MGO_EINVAL;
    const level_t *L = &s->lv[level];
    if (wx) memcpy(wx, L->wx, (size_t)L->ny * L->nz * sizeof(double));
    if (wy) memcpy(wy, L->wy, (size_t)L->nx * L->nz * sizeof(double));
    if (wz) memcpy(wz, L->wz, (size_t)L->nx * L->ny * sizeof(double));
    return MGO_OK;
}

int mgo_get_faces(const mgo_solver *s, int level, double *bx, double *by, double *bz)
{
    if (!s || level < 0 || level >= s->nlev) return MGO_EINVAL;
    const level_t *L = &s->lv[level];
    size_t bytes = lv_cells(L) * sizeof(double);
    if (bx) memcpy(bx, L->bx, bytes);
    if (by) memcpy(by, L->by, bytes);
    if (bz) memcpy(bz, L->bz, bytes);
    return MGO_OK;
}

int mgo_apply(const mgo_solver *s, int level, const double *p, double *out)
{
    if (!s || level < 0 || level >= s->nlev || !p || !out) return MGO_EINVAL;
    apply(&s->lv[level], p, out);
    return MGO_OK;
}

int mgo_smooth_half(const mgo_solver *s, int level, int colour, const double *f, double *p)
{
    if (!s || level < 0 || level >= s->nlev || (colour != 0 && colour != 1) || !f || !p)
        return MGO_EINVAL;
    smooth_half(&s->lv[level], colour, f, p);
    return MGO_OK;
}

int mgo_residual_level(const mgo_solver *s, int level, const double *f, const double *p, double *r)
{
    if (!s || level < 0 || level >= s->nlev || !f || !p || !r) return MGO_EINVAL;
    residual(&s->lv[level], f, p, r);
    return MGO_OK;
}

int mgo_restrict(const mgo_solver *s, int level, const double *r, double *fc)
{
    if (!s || level < 0 || level >= s->nlev - 1 || !r || !fc) return MGO_EINVAL;
    restrict8(&s->lv[level], &s->lv[level + 1], r, fc);
    return MGO_OK;
}

int mgo_prolong_add(const mgo_solver *s, int level, const double *e, double *p)
{
    if (!s || level < 0 || level >= s->nlev - 1 || !e || !p) return MGO_EINVAL;
    prolong_add(s, &s->lv[level], &s->lv[level + 1], e, p);
    return MGO_OK;
}
