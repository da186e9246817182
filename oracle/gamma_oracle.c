/*
 * gamma_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU implementation of what the gamma-index
 * hot path computes (arxiv/paper_1012_1900, Gu, Jia, Jiang, "GPU-based fast gamma
 * index calculation").  It exists so that the CUDA path can be compared against
 * something written straight from the paper.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with paper_1012_1900_b200/csrc.
 *
 * What it computes (section 2.1, Eq. 1; readings in DESIGN.md):
 *
 *   gamma(r_r) = min over the continuous evaluation surface of
 *                | (r_r/dd , D_r(r_r)/dD) - (r_e/dd , D_e(r_e)/dD) |
 *
 * where the evaluation surface is the piecewise-linear interpolant of the
 * evaluation dose grid: every grid cell is Kuhn-split into n! simplices
 * (vertex chain c, c+e_p(1), c+e_p(1)+e_p(2), ... for each permutation p) and
 * "the accurate Gamma can be obtained by calculating the distance from the
 * reference point to the continuous evaluation surface formed by discrete
 * evaluation points" (citing Ju et al. 2008).
 *
 * The point-to-simplex distance follows PAPER.md:204-207 literally:
 *   {w_1..w_k} = (V^T V)^-1 V^T P,  w_{k+1} = 1 - sum w_i,
 * evaluated on EVERY non-empty vertex subset of the simplex ("we calculate
 * Gamma in all simplexes") and keeping the feasible (all weights
 * >= 0) candidates.  A second, independent routine implements the recursion the
 * paper attributes to Ju et al. (recurse only into the facets
 * opposite negative weights); tests check the two agree.
 *
 * Search region: "a search range of a radius (DD(r_r)/dD) dd":
 * only cells whose minimum spatial distance L_cell is below gamma_0 = |DD|/dD
 * can matter.  Two forms are provided (reading 3/4):
 *   form 0 "plain": every in-grid cell with L_cell < gamma_0;
 *   form 1 "shell": Chebyshev shells s = 0,1,2,... around the voxel, stopping at
 *           the first shell whose smallest possible L_cell is >= the current best
 *           (same visits as Algorithm A1 steps 4-b with the break read as
 *           "L_n >= gamma", reading 3).
 * They give the same minimum.
 *
 * Parity pins (tests/test_oracle_pins.py): identical grids -> 0; flat fields with
 * offset c -> |c|/dD; linear ramp closed form; gamma(k dD, k dd) = gamma/k; axis
 * permutation invariance; brute-force barycentric sampling on tiny grids; 1D
 * polyline by hand; plain == shell; all-subsets == Ju recursion;
 * gamma_interp <= gamma_vertex_only.
 * Since round 3 also against EXACT rational arithmetic, voxel by voxel
 * (tests/test_exact_pins.py, tests/exact_gamma.py): equal to 1e-11.
 * Parity UNPINNED by the paper (conventions only, readings 6, 8-10):
 * orientation of the Kuhn diagonal; cutoff / local-mode / NaN policy.
 *
 * VALIDITY LIMIT (reading 21).  The normal equations square the
 * condition number of V.  Under the local criterion a reference dose D_r that
 * is tiny against the evaluation doses around it (dD_v = DD * D_r) stretches the
 * dose axis by s ~ |D_e - D_r| / dD_v; the Gram matrix then has a condition
 * number ~ s^2 and at s ~ 1e8 and beyond double precision has no digits left:
 * this oracle then returns the distance to a point of the surface that is not
 * the closest one (an OVER-estimate; measured 0.5 above the exact value at
 * D_r = 1e-10).  It is trusted, and compared with the CUDA path, where
 * D_r >= 1e-4 D_norm; below that the tests use exact arithmetic instead.
 * Nothing in the arithmetic of this file was changed for it.
 *
 * Layout: dense, x fastest: lin = ix + nx*(iy + ny*iz).  An axis of size 1 is
 * dropped (reading 12).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAXDIM 4 /* n+1 with n <= 3 */

/* ---------------------------------------------------------------------- */
/* small dense helpers (sizes <= 3)                                        */
/* ---------------------------------------------------------------------- */

/* Solve the SPD system G w = b (size m <= 3) by Cholesky.  Returns 0 on
 * success, 1 if G is not positive definite. */
static int chol_solve(int m, const double G[3][3], const double b[3], double w[3])
{
    double Lc[3][3];
    memset(Lc, 0, sizeof Lc);
    for (int i = 0; i < m; ++i) {
        for (int j = 0; j <= i; ++j) {
            double s = G[i][j];
            for (int k = 0; k < j; ++k) s -= Lc[i][k] * Lc[j][k];
            if (i == j) {
                if (!(s > 0.0)) return 1;
                Lc[i][i] = sqrt(s);
            } else {
                Lc[i][j] = s / Lc[j][j];
            }
        }
    }
    double y[3];
    for (int i = 0; i < m; ++i) {
        double s = b[i];
        for (int k = 0; k < i; ++k) s -= Lc[i][k] * y[k];
        y[i] = s / Lc[i][i];
    }
    for (int i = m - 1; i >= 0; --i) {
        double s = y[i];
        for (int k = i + 1; k < m; ++k) s -= Lc[k][i] * w[k];
        w[i] = s / Lc[i][i];
    }
    return 0;
}

/* Projection of the origin onto the affine hull of the points q[idx[0..nv-1]]
 * (each a K-vector, row-major in q).  PAPER.md:204-207: the last listed vertex
 * plays the role of v_{k+1}; P = (reference point) - v_{k+1} = -v_{k+1};
 * V's columns are v_i - v_{k+1}.  Writes the nv barycentric weights and returns
 * the distance |P - V w|.  Returns -1 if the normal equations are singular. */
static double affine_projection(const double *q, int K, const int *idx, int nv, double *wout)
{
    const double *base = q + (size_t)idx[nv - 1] * K;
    int m = nv - 1;
    double V[3][ORACLE_MAXDIM], P[ORACLE_MAXDIM];
    for (int c = 0; c < K; ++c) P[c] = 0.0 - base[c];
    for (int i = 0; i < m; ++i)
        for (int c = 0; c < K; ++c) V[i][c] = q[(size_t)idx[i] * K + c] - base[c];
    double w[3] = {0, 0, 0};
    if (m > 0) {
        double G[3][3], b[3];
        for (int i = 0; i < m; ++i) {
            for (int j = 0; j < m; ++j) {
                double s = 0.0;
                for (int c = 0; c < K; ++c) s += V[i][c] * V[j][c];
                G[i][j] = s;
            }
            double s = 0.0;
            for (int c = 0; c < K; ++c) s += V[i][c] * P[c];
            b[i] = s;
        }
        if (chol_solve(m, G, b, w)) return -1.0;
    }
    double sumw = 0.0, r2 = 0.0;
    for (int i = 0; i < m; ++i) sumw += w[i];
    for (int c = 0; c < K; ++c) {
        double r = P[c];
        for (int i = 0; i < m; ++i) r -= V[i][c] * w[i];
        r2 += r * r;
    }
    for (int i = 0; i < m; ++i) wout[i] = w[i];
    wout[m] = 1.0 - sumw;
    return sqrt(r2);
}

/* Distance from the origin to the simplex conv{q_0..q_{nv-1}} in R^K by the
 * "all simplexes" formulation: every non-empty vertex subset is
 * projected; a subset whose weights are all >= 0 contributes its distance. */
double oracle_simplex_distance(const double *q, int nv, int K)
{
    double best = INFINITY;
    for (unsigned mask = 1; mask < (1u << nv); ++mask) {
        int idx[ORACLE_MAXDIM], c = 0;
        for (int i = 0; i < nv; ++i)
            if (mask & (1u << i)) idx[c++] = i;
        double w[ORACLE_MAXDIM];
        double d = affine_projection(q, K, idx, c, w);
        if (d < 0.0) continue;
        int ok = 1;
        for (int i = 0; i < c; ++i)
            if (!(w[i] >= 0.0)) ok = 0;
        if (ok && d < best) best = d;
    }
    return best;
}

/* Second, independent algorithm: the recursion of Ju et al. as described in
 * project on the whole simplex; if some weights are negative,
 * recurse only into the facets opposite those vertices. */
static double ju_rec(const double *q, int K, const int *idx, int nv)
{
    double w[ORACLE_MAXDIM];
    double d = affine_projection(q, K, idx, nv, w);
    if (nv == 1) return d;
    int anyneg = 0;
    double best = INFINITY;
    if (d >= 0.0) {
        for (int i = 0; i < nv; ++i)
            if (w[i] < 0.0) anyneg = 1;
        if (!anyneg) return d;
    }
    for (int i = 0; i < nv; ++i) {
        if (d >= 0.0 && !(w[i] < 0.0)) continue;
        int sub[ORACLE_MAXDIM], c = 0;
        for (int j = 0; j < nv; ++j)
            if (j != i) sub[c++] = idx[j];
        double s = ju_rec(q, K, sub, c);
        if (s < best) best = s;
    }
    return best;
}

double oracle_simplex_distance_ju(const double *q, int nv, int K)
{
    int idx[ORACLE_MAXDIM];
    for (int i = 0; i < nv; ++i) idx[i] = i;
    return ju_rec(q, K, idx, nv);
}

/* ---------------------------------------------------------------------- */
/* the gamma search                                                        */
/* ---------------------------------------------------------------------- */

typedef struct {
    int n;            /* number of active axes (size > 1) */
    int ax[3];        /* which of x,y,z they are */
    long long dim[3]; /* sizes of the active axes */
    long long str[3]; /* linear strides of the active axes */
    double hn[3];     /* spacing / DTA of the active axes */
} grid_t;

static const int PERM1[1][3] = {{0, 0, 0}};
static const int PERM2[2][3] = {{0, 1, 0}, {1, 0, 0}};
static const int PERM3[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};

/* minimum spatial distance (normalised by DTA) from the voxel to the cell at
 * integer offset o (cell = [o, o+1] per axis): DESIGN.md reading 4. */
static double cell_bound(const grid_t *g, const long long *o)
{
    double s = 0.0;
    for (int a = 0; a < g->n; ++a) {
        long long m = o[a] > -o[a] - 1 ? o[a] : -o[a] - 1;
        if (m < 0) m = 0;
        double d = (double)m * g->hn[a];
        s += d * d;
    }
    return sqrt(s);
}

/* distance from the reference point of voxel v to the n! Kuhn simplices of the
 * in-grid cell whose minimum corner is c = v + o. */
static double cell_distance(const grid_t *g, const double *eval, const long long *v, const long long *o,
                            double Dr, double dD)
{
    int n = g->n, K = n + 1;
    int nperm = n == 3 ? 6 : (n == 2 ? 2 : 1);
    const int(*perm)[3] = n == 3 ? PERM3 : (n == 2 ? PERM2 : PERM1);
    double best = INFINITY;
    for (int p = 0; p < nperm; ++p) {
        double q[ORACLE_MAXDIM * ORACLE_MAXDIM];
        long long u[3];
        for (int a = 0; a < n; ++a) u[a] = v[a] + o[a];
        for (int m = 0; m <= n; ++m) {
            if (m > 0) u[perm[p][m - 1]] += 1;
            long long lin = 0;
            for (int a = 0; a < n; ++a) {
                q[m * K + a] = (double)(u[a] - v[a]) * g->hn[a];
                lin += u[a] * g->str[a];
            }
            q[m * K + n] = (eval[lin] - Dr) / dD;
        }
        double d = oracle_simplex_distance(q, n + 1, K);
        if (d < best) best = d;
    }
    return best;
}

static int cell_in_grid(const grid_t *g, const long long *v, const long long *o)
{
    for (int a = 0; a < g->n; ++a) {
        long long c = v[a] + o[a];
        if (c < 0 || c > g->dim[a] - 2) return 0;
    }
    return 1;
}

static double gamma_plain(const grid_t *g, const double *eval, const long long *v, double Dr, double dD,
                          double g0)
{
    double best = g0;
    long long lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, o[3] = {0, 0, 0};
    for (int a = 0; a < g->n; ++a) {
        long long r = (long long)ceil(g0 / g->hn[a]) + 1;
        lo[a] = -r - 1;
        hi[a] = r;
    }
    for (o[2] = lo[2]; o[2] <= hi[2]; ++o[2])
        for (o[1] = lo[1]; o[1] <= hi[1]; ++o[1])
            for (o[0] = lo[0]; o[0] <= hi[0]; ++o[0]) {
                if (!cell_in_grid(g, v, o)) continue;
                if (!(cell_bound(g, o) < g0)) continue;
                double d = cell_distance(g, eval, v, o, Dr, dD);
                if (d < best) best = d;
            }
    return best;
}

static double gamma_shell(const grid_t *g, const double *eval, const long long *v, double Dr, double dD,
                          double g0)
{
    double best = g0;
    double hmin = g->hn[0];
    for (int a = 1; a < g->n; ++a)
        if (g->hn[a] < hmin) hmin = g->hn[a];
    long long maxdim = 0;
    for (int a = 0; a < g->n; ++a)
        if (g->dim[a] > maxdim) maxdim = g->dim[a];
    for (long long s = 0; s <= maxdim; ++s) {
        if ((double)s * hmin >= best) break;
        long long lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, o[3] = {0, 0, 0};
        for (int a = 0; a < g->n; ++a) {
            lo[a] = -s - 1;
            hi[a] = s;
        }
        for (o[2] = lo[2]; o[2] <= hi[2]; ++o[2])
            for (o[1] = lo[1]; o[1] <= hi[1]; ++o[1])
                for (o[0] = lo[0]; o[0] <= hi[0]; ++o[0]) {
                    long long cheb = 0;
                    for (int a = 0; a < g->n; ++a) {
                        long long m = o[a] > -o[a] - 1 ? o[a] : -o[a] - 1;
                        if (m > cheb) cheb = m;
                    }
                    if (cheb != s) continue;
                    if (!cell_in_grid(g, v, o)) continue;
                    if (!(cell_bound(g, o) < best)) continue;
                    double d = cell_distance(g, eval, v, o, Dr, dD);
                    if (d < best) best = d;
                }
    }
    return best;
}

/* classical discrete search: minimum over evaluation GRID POINTS only (no
 * interpolation), exhaustive inside the radius gamma_0.  Used only as a pin:
 * gamma_interp <= gamma_vertex_only. */
static double gamma_vertex_only(const grid_t *g, const double *eval, const long long *v, double Dr,
                                double dD, double g0)
{
    double best = g0;
    long long lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, o[3] = {0, 0, 0};
    for (int a = 0; a < g->n; ++a) {
        long long r = (long long)ceil(g0 / g->hn[a]);
        lo[a] = -r;
        hi[a] = r;
    }
    for (o[2] = lo[2]; o[2] <= hi[2]; ++o[2])
        for (o[1] = lo[1]; o[1] <= hi[1]; ++o[1])
            for (o[0] = lo[0]; o[0] <= hi[0]; ++o[0]) {
                long long lin = 0;
                int ok = 1;
                double s2 = 0.0;
                for (int a = 0; a < g->n; ++a) {
                    long long u = v[a] + o[a];
                    if (u < 0 || u >= g->dim[a]) ok = 0;
                    lin += u * g->str[a];
                    double d = (double)o[a] * g->hn[a];
                    s2 += d * d;
                }
                if (!ok) continue;
                double dd = (eval[lin] - Dr) / dD;
                double d = sqrt(s2 + dd * dd);
                if (d < best) best = d;
            }
    return best;
}

static long long count_visits(const grid_t *g, const long long *v, double gam)
{
    long long lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, o[3] = {0, 0, 0}, cnt = 0;
    for (int a = 0; a < g->n; ++a) {
        long long r = (long long)ceil(gam / g->hn[a]) + 1;
        lo[a] = -r - 1;
        hi[a] = r;
    }
    for (o[2] = lo[2]; o[2] <= hi[2]; ++o[2])
        for (o[1] = lo[1]; o[1] <= hi[1]; ++o[1])
            for (o[0] = lo[0]; o[0] <= hi[0]; ++o[0])
                if (cell_in_grid(g, v, o) && cell_bound(g, o) < gam) ++cnt;
    return cnt;
}

/*
 * oracle_gamma
 *   ref, eval   : N = nx*ny*nz doubles (the fp32 inputs widened exactly), x fastest
 *   dims        : (nx, ny, nz); spacing_mm > 0
 *   DD          : dose-difference criterion as a fraction; DTA_mm > 0
 *   mode        : 0 global (dD = DD * D_norm), 1 local (dD_v = DD * D_r[v])
 *   cutoff      : voxels with D_r < cutoff * D_norm are excluded (NaN)
 *   norm_dose   : D_norm; <= 0 means max(ref)
 *   form        : 0 plain radius, 1 shell, 2 vertex-only (pin only)
 *   vox_list    : NULL -> all N voxels, out_gamma has N entries (lin index order);
 *                 else n_list linear voxel indices, out_gamma has n_list entries
 *   out_visits  : optional; N_s(v) = #in-grid cells with L_cell < gamma[v]
 *   nthreads    : OpenMP threads (<=0: default)
 * returns 0, or 1 on invalid arguments.
 */
int oracle_gamma(const double *ref, const double *eval, const int dims[3], const double spacing_mm[3],
                 double DD, double DTA_mm, int mode, double cutoff, double norm_dose, int form,
                 const long long *vox_list, long long n_list, double *out_gamma, long long *out_visits,
                 int nthreads)
{
    if (!ref || !eval || !out_gamma || !(DD > 0.0) || !(DTA_mm > 0.0)) return 1;
    if (mode != 0 && mode != 1) return 1;
    if (!(cutoff >= 0.0 && cutoff < 1.0)) return 1;
    grid_t g;
    memset(&g, 0, sizeof g);
    long long N = 1, stride = 1;
    for (int a = 0; a < 3; ++a) {
        if (dims[a] < 1 || !(spacing_mm[a] > 0.0)) return 1;
        if (dims[a] > 1) {
            g.ax[g.n] = a;
            g.dim[g.n] = dims[a];
            g.str[g.n] = stride;
            g.hn[g.n] = spacing_mm[a] / DTA_mm;
            g.n++;
        }
        stride *= dims[a];
        N *= dims[a];
    }
    if (g.n < 1) return 1;
    double dnorm = norm_dose;
    if (!(dnorm > 0.0)) {
        dnorm = ref[0];
        for (long long i = 1; i < N; ++i)
            if (ref[i] > dnorm) dnorm = ref[i];
    }
    long long count = vox_list ? n_list : N;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
    for (long long t = 0; t < count; ++t) {
        long long lin = vox_list ? vox_list[t] : t;
        double Dr = ref[lin];
        double dD = mode == 0 ? DD * dnorm : DD * Dr;
        if (out_visits) out_visits[t] = 0;
        if (Dr < cutoff * dnorm || !(dD > 0.0)) {
            out_gamma[t] = NAN;
            continue;
        }
        long long v[3] = {0, 0, 0}, rem = lin;
        {
            long long full[3];
            for (int a = 0; a < 3; ++a) {
                full[a] = rem % dims[a];
                rem /= dims[a];
            }
            for (int a = 0; a < g.n; ++a) v[a] = full[g.ax[a]];
        }
        double g0 = fabs(eval[lin] - Dr) / dD; /* A1 step 4a */
        double gam;
        if (form == 0)
            gam = gamma_plain(&g, eval, v, Dr, dD, g0);
        else if (form == 1)
            gam = gamma_shell(&g, eval, v, Dr, dD, g0);
        else
            gam = gamma_vertex_only(&g, eval, v, Dr, dD, g0);
        out_gamma[t] = gam;
        if (out_visits) out_visits[t] = count_visits(&g, v, gam);
    }
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
