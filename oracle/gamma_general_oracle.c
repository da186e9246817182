/*
 * gamma_general_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU definition of the gamma index when the evaluation dose lives on ITS OWN grid
 * (dims, spacing, origin different from the reference grid's), with the closest point of the evaluation surface as a
 * second output.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code, header, table or helper with
 * paper_1012_1900_b200/csrc -- nor with gamma_oracle.c, which stays as pinned in round 1.
 *
 * What it computes (section 2.1, Eq. 1):
 *
 *   gamma(r_r) = min over r_e of sqrt( |r_r - r_e|^2 / dd^2 + (D_r(r_r) - D_e(r_e))^2 / dD^2 )
 *
 * with r_e ranging over the CONTINUOUS evaluation surface: the piecewise-linear interpolant of the
 * evaluation grid on the Kuhn split of its cells (readings 5, 6 of DESIGN.md).  The paper's data put both doses on
 * one grid but Eq. 1 does not need that: here the reference point of voxel v sits at
 *   r_r = ref_origin + v * ref_spacing        (mm, per axis)
 * and evaluation vertex u at  eval_origin + u * eval_spacing.  The refinements the paper cites (PAPER.md:135,
 * Stock et al. 2005: the "gamma angle", i.e. which of dose difference and distance dominates) need the point where
 * the minimum is attained: closest[4] = (x, y, z in mm, interpolated evaluation dose) of one minimiser.
 *
 * VALIDITY LIMIT (reading 21), as for gamma_oracle.c: under the local criterion with a reference dose far
 * below the evaluation doses around it the Gram matrix is too ill conditioned for double precision and the result is an
 * over-estimate; trusted where D_r >= 1e-4 D_norm (tests/test_exact_pins.py).
 *
 * Point-to-simplex distance: PAPER.md:204-207 literally -- {w} = (V^T V)^-1 V^T P, w_{k+1} = 1 - sum w -- on EVERY
 * non-empty vertex subset of the simplex, feasible candidates (all weights >= 0) kept; the weights of
 * the winning candidate give the closest point.
 *
 * Search region.  form 0 "all": every cell of the evaluation grid, no pruning at all (the definition; tiny grids).
 * form 1 "shell": cells in Chebyshev shells s = 0, 1, 2, ... around the evaluation cell that holds (or is nearest to)
 * the reference point, visited only if the cell's exact minimum spatial distance to the point is below the running
 * minimum; stops at the first shell none of whose cells can be closer (every cell of shell s >= 1 is at least
 * (s - 1) * min spacing / dd away: reading 4 of DESIGN.md carried over to a point that is not a grid vertex).
 * The two forms give the same gamma (tests).
 *
 * Exclusion policy as in gamma_oracle.c (readings 8-10): D_norm = max(ref) unless given; excluded (NaN) if
 * D_r < cutoff * D_norm or dD_v <= 0.  Axes: all three must be active on the evaluation grid (size >= 2); a
 * reference grid may have any dims >= 1.
 *
 * Pins (tests/test_general_oracle_pins.py): an integer-voxel origin shift equals an index shift of the same-grid
 * oracle; identical geometry equals gamma_oracle.c bit for bit; linear-ramp closed form with unequal spacings and a
 * fractional origin offset; brute force with a library QP over all simplices of tiny grids; the closest point is on
 * the surface and its normalised distance is gamma; form 0 == form 1.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- dense helpers for systems of size <= 3 -------------------------------------------------------------------- */

/* Gaussian elimination with partial pivoting; returns 0 on success, 1 if singular. */
static int solve_small(int m, double A[3][3], double b[3], double x[3])
{
    int piv[3] = {0, 1, 2};
    for (int c = 0; c < m; ++c) {
        int best = c;
        for (int r = c + 1; r < m; ++r)
            if (fabs(A[piv[r]][c]) > fabs(A[piv[best]][c])) best = r;
        int t = piv[c]; piv[c] = piv[best]; piv[best] = t;
        double p = A[piv[c]][c];
        if (!(fabs(p) > 0.0)) return 1;
        for (int r = c + 1; r < m; ++r) {
            double f = A[piv[r]][c] / p;
            for (int k = c; k < m; ++k) A[piv[r]][k] -= f * A[piv[c]][k];
            b[piv[r]] -= f * b[piv[c]];
        }
    }
    for (int c = m - 1; c >= 0; --c) {
        double s = b[piv[c]];
        for (int k = c + 1; k < m; ++k) s -= A[piv[c]][k] * x[k];
        x[c] = s / A[piv[c]][c];
    }
    return 0;
}

/* Distance from the origin to conv{q_0..q_3} in R^4 (rows of q) by projecting on every vertex subset; weights of the
 * winner are written to wbest (zeros for vertices not in the winning subset). */
static double simplex_distance_weights(const double q[4][4], double wbest[4])
{
    double best = INFINITY;
    for (unsigned mask = 1; mask < 16; ++mask) {
        int idx[4], nv = 0;
        for (int i = 0; i < 4; ++i)
            if (mask & (1u << i)) idx[nv++] = i;
        const double *base = q[idx[nv - 1]];
        int m = nv - 1;
        double V[3][4], P[4], w[3] = {0, 0, 0};
        for (int c = 0; c < 4; ++c) P[c] = -base[c];
        for (int i = 0; i < m; ++i)
            for (int c = 0; c < 4; ++c) V[i][c] = q[idx[i]][c] - base[c];
        if (m > 0) {
            double G[3][3], rhs[3];
            for (int i = 0; i < m; ++i) {
                for (int j = 0; j < m; ++j) {
                    double s = 0.0;
                    for (int c = 0; c < 4; ++c) s += V[i][c] * V[j][c];
                    G[i][j] = s;
                }
                double s = 0.0;
                for (int c = 0; c < 4; ++c) s += V[i][c] * P[c];
                rhs[i] = s;
            }
            if (solve_small(m, G, rhs, w)) continue;
        }
        double sumw = 0.0, r2 = 0.0;
        int ok = 1;
        for (int i = 0; i < m; ++i) {
            sumw += w[i];
            if (!(w[i] >= 0.0)) ok = 0;
        }
        if (!(1.0 - sumw >= 0.0)) ok = 0;
        if (!ok) continue;
        for (int c = 0; c < 4; ++c) {
            double r = P[c];
            for (int i = 0; i < m; ++i) r -= V[i][c] * w[i];
            r2 += r * r;
        }
        double d = sqrt(r2);
        if (d < best) {
            best = d;
            for (int i = 0; i < 4; ++i) wbest[i] = 0.0;
            for (int i = 0; i < m; ++i) wbest[idx[i]] = w[i];
            wbest[idx[nv - 1]] = 1.0 - sumw;
        }
    }
    return best;
}

typedef struct {
    long long n[3];  /* evaluation grid dims */
    double h[3];     /* evaluation spacing / DTA */
} egrid_t;

static const int PERM[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};

/* All six Kuhn tetrahedra of evaluation cell c against the reference point at fractional evaluation index u.
 * Updates *best and, when improved, the closest point (fractional evaluation index + dose). */
static void cell_update(const egrid_t *g, const double *eval, const long long c[3], const double u[3], double Dr,
                        double dD, double *best, double closest_idx[3], double *closest_dose)
{
    for (int p = 0; p < 6; ++p) {
        double q[4][4], dose[4];
        long long vtx[4][3];
        long long cur[3] = {c[0], c[1], c[2]};
        for (int m = 0; m < 4; ++m) {
            if (m > 0) cur[PERM[p][m - 1]] += 1;
            for (int a = 0; a < 3; ++a) {
                vtx[m][a] = cur[a];
                q[m][a] = ((double)cur[a] - u[a]) * g->h[a];
            }
            dose[m] = eval[cur[0] + g->n[0] * (cur[1] + g->n[1] * cur[2])];
            q[m][3] = (dose[m] - Dr) / dD;
        }
        double w[4];
        double d = simplex_distance_weights(q, w);
        if (d < *best) {
            *best = d;
            for (int a = 0; a < 3; ++a) {
                double s = 0.0;
                for (int m = 0; m < 4; ++m) s += w[m] * (double)vtx[m][a];
                closest_idx[a] = s;
            }
            double s = 0.0;
            for (int m = 0; m < 4; ++m) s += w[m] * dose[m];
            *closest_dose = s;
        }
    }
}

/* exact minimum spatial distance (normalised) from the point at fractional index u to the cell [c, c+1]^3 */
static double cell_bound(const egrid_t *g, const long long c[3], const double u[3])
{
    double s = 0.0;
    for (int a = 0; a < 3; ++a) {
        double lo = (double)c[a] - u[a], hi = u[a] - (double)(c[a] + 1);
        double d = lo > hi ? lo : hi;
        if (d < 0.0) d = 0.0;
        d *= g->h[a];
        s += d * d;
    }
    return sqrt(s);
}

/*
 * oracle_gamma_general
 *   ref            : ref_dims[0]*ref_dims[1]*ref_dims[2] doubles, x fastest
 *   ref_dims/ref_spacing_mm/ref_origin_mm  : reference grid; the centre of voxel (i,j,k) is origin + (i,j,k)*spacing
 *   eval, eval_dims/eval_spacing_mm/eval_origin_mm : evaluation grid, every dim >= 2
 *   DD, DTA_mm, mode, cutoff, norm_dose : as oracle_gamma
 *   form           : 0 every cell of the evaluation grid, 1 shells with the exact cell bound
 *   vox_list       : NULL -> all reference voxels; else n_list linear reference-voxel indices
 *   out_gamma      : count doubles (NaN = excluded)
 *   out_closest    : optional, count x 4 doubles: x, y, z (mm) and evaluation dose of one closest surface point
 * returns 0, or 1 on invalid arguments.
 */
int oracle_gamma_general(const double *ref, const int ref_dims[3], const double ref_spacing_mm[3],
                         const double ref_origin_mm[3], const double *eval, const int eval_dims[3],
                         const double eval_spacing_mm[3], const double eval_origin_mm[3], double DD, double DTA_mm,
                         int mode, double cutoff, double norm_dose, int form, const long long *vox_list,
                         long long n_list, double *out_gamma, double *out_closest, int nthreads)
{
    if (!ref || !eval || !out_gamma || !(DD > 0.0) || !(DTA_mm > 0.0)) return 1;
    if (mode != 0 && mode != 1) return 1;
    if (!(cutoff >= 0.0 && cutoff < 1.0)) return 1;
    if (form != 0 && form != 1) return 1;
    egrid_t g;
    long long Nr = 1;
    for (int a = 0; a < 3; ++a) {
        if (ref_dims[a] < 1 || eval_dims[a] < 2) return 1;
        if (!(ref_spacing_mm[a] > 0.0) || !(eval_spacing_mm[a] > 0.0)) return 1;
        g.n[a] = eval_dims[a];
        g.h[a] = eval_spacing_mm[a] / DTA_mm;
        Nr *= ref_dims[a];
    }
    double hmin = g.h[0] < g.h[1] ? g.h[0] : g.h[1];
    if (g.h[2] < hmin) hmin = g.h[2];
    long long maxdim = g.n[0] > g.n[1] ? g.n[0] : g.n[1];
    if (g.n[2] > maxdim) maxdim = g.n[2];
    double dnorm = norm_dose;
    if (!(dnorm > 0.0)) {
        dnorm = ref[0];
        for (long long i = 1; i < Nr; ++i)
            if (ref[i] > dnorm) dnorm = ref[i];
    }
    long long count = vox_list ? n_list : Nr;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (long long t = 0; t < count; ++t) {
        long long lin = vox_list ? vox_list[t] : t;
        double Dr = ref[lin];
        double dD = mode == 0 ? DD * dnorm : DD * Dr;
        if (out_closest)
            for (int k = 0; k < 4; ++k) out_closest[4 * t + k] = NAN;
        if (Dr < cutoff * dnorm || !(dD > 0.0)) {
            out_gamma[t] = NAN;
            continue;
        }
        long long v[3], rem = lin;
        for (int a = 0; a < 3; ++a) {
            v[a] = rem % ref_dims[a];
            rem /= ref_dims[a];
        }
        double u[3]; /* the reference point in fractional evaluation-index coordinates */
        long long c0[3];
        for (int a = 0; a < 3; ++a) {
            double x = ref_origin_mm[a] + (double)v[a] * ref_spacing_mm[a];
            u[a] = (x - eval_origin_mm[a]) / eval_spacing_mm[a];
            double f = floor(u[a]);
            long long c = (long long)f;
            if (c < 0) c = 0;
            if (c > g.n[a] - 2) c = g.n[a] - 2;
            c0[a] = c;
        }
        double best = INFINITY, cidx[3] = {0, 0, 0}, cdose = 0.0;
        if (form == 0) {
            long long c[3];
            for (c[2] = 0; c[2] <= g.n[2] - 2; ++c[2])
                for (c[1] = 0; c[1] <= g.n[1] - 2; ++c[1])
                    for (c[0] = 0; c[0] <= g.n[0] - 2; ++c[0]) cell_update(&g, eval, c, u, Dr, dD, &best, cidx, &cdose);
        } else {
            for (long long s = 0; s <= maxdim; ++s) {
                if (s >= 1 && (double)(s - 1) * hmin >= best) break;
                long long o[3], c[3];
                for (o[2] = -s; o[2] <= s; ++o[2])
                    for (o[1] = -s; o[1] <= s; ++o[1])
                        for (o[0] = -s; o[0] <= s; ++o[0]) {
                            long long cheb = 0;
                            int in = 1;
                            for (int a = 0; a < 3; ++a) {
                                long long m = o[a] < 0 ? -o[a] : o[a];
                                if (m > cheb) cheb = m;
                                c[a] = c0[a] + o[a];
                                if (c[a] < 0 || c[a] > g.n[a] - 2) in = 0;
                            }
                            if (cheb != s || !in) continue;
                            if (!(cell_bound(&g, c, u) < best)) continue;
                            cell_update(&g, eval, c, u, Dr, dD, &best, cidx, &cdose);
                        }
            }
        }
        out_gamma[t] = best;
        if (out_closest) {
            for (int a = 0; a < 3; ++a) out_closest[4 * t + a] = eval_origin_mm[a] + cidx[a] * eval_spacing_mm[a];
            out_closest[4 * t + 3] = cdose;
        }
    }
    return 0;
}
