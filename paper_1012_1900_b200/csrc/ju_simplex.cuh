// ju_simplex.cuh -- the paper's own point-to-simplex routine as a kernel VARIANT (opts.interpolation = 3):
// projection onto the affine hull through the normal equations (V^T V) w = V^T P, w_{k+1} = 1 - sum w
// (PAPER.md:204-207), and, when a weight is negative, recursion into the sub-simplices opposite the negative
// weights only (Ju et al.) -- instead of the paper's GPU choice of evaluating ALL sub-simplices
// and instead of this library's default closed form on owned faces (features_generated.cuh).
// Same evaluation surface (Kuhn split of every grid cell), same result up to rounding; branchy and an order of
// magnitude slower: it exists to measure that trade, not to be fast.
//
// Exactness of the recursion: if every facet containing the closest point had a non-negative weight at the
// projection p, moving from the closest point toward p would stay inside the simplex -- a contradiction; so the
// closest point lies in a facet opposite a negative weight.
#pragma once
#include "common.cuh"

namespace gamma_b200 {

// Squared distance from the origin to the simplex spanned by the vertices of q selected by the bits of `full`
// (up to 4 vertices in R^4).  Iterative form of the recursion: a stack of vertex subsets, each visited once.
__device__ inline float ju_simplex_dist2(const float (&q)[4][4], unsigned full)
{
    float best = INFINITY;
    unsigned visited = 0u;                       // bit m: subset m was expanded
    unsigned stack[16];
    int sp = 0;
    stack[sp++] = full;
    while (sp > 0) {
        const unsigned m = stack[--sp];
        if ((visited >> m) & 1u) continue;
        visited |= 1u << m;
        int idx[4], n = 0;
#pragma unroll
        for (int s = 0; s < 4; ++s)
            if ((m >> s) & 1u) idx[n++] = s;
        const float* qb = q[idx[0]];             // base vertex b: P = -q_b, V = [q_s - q_b]
        if (n == 1) {
            best = fminf(best, qb[0] * qb[0] + qb[1] * qb[1] + qb[2] * qb[2] + qb[3] * qb[3]);
            continue;
        }
        const int k = n - 1;
        float E[3][4], G[3][3], rhs[3], t[3];
        for (int i = 0; i < k; ++i) {
            float r = 0.0f;
            for (int c = 0; c < 4; ++c) {
                E[i][c] = q[idx[i + 1]][c] - qb[c];
                r = fmaf(-E[i][c], qb[c], r);
            }
            rhs[i] = r;
        }
        for (int i = 0; i < k; ++i)
            for (int j = 0; j <= i; ++j) {
                float s = 0.0f;
                for (int c = 0; c < 4; ++c) s = fmaf(E[i][c], E[j][c], s);
                G[i][j] = s;
            }
        // Cholesky G = L L^T in place (SPD: the spatial parts of Kuhn edges are linearly independent), then the
        // two triangular solves
        for (int i = 0; i < k; ++i) {
            for (int j = 0; j <= i; ++j) {
                float s = G[i][j];
                for (int l = 0; l < j; ++l) s = fmaf(-G[i][l], G[j][l], s);
                G[i][j] = (i == j) ? sqrtf(fmaxf(s, 1e-30f)) : s / G[j][j];
            }
        }
        for (int i = 0; i < k; ++i) {
            float s = rhs[i];
            for (int l = 0; l < i; ++l) s = fmaf(-G[i][l], t[l], s);
            t[i] = s / G[i][i];
        }
        for (int i = k - 1; i >= 0; --i) {
            float s = t[i];
            for (int l = i + 1; l < k; ++l) s = fmaf(-G[l][i], t[l], s);
            t[i] = s / G[i][i];
        }
        float wb = 1.0f;
        bool feasible = true;
        for (int i = 0; i < k; ++i) { wb -= t[i]; feasible = feasible && t[i] >= 0.0f; }
        feasible = feasible && wb >= 0.0f;
        if (feasible) {                          // foot point inside: explicit residual q_b + sum t_i E_i
            float d2 = 0.0f;
            for (int c = 0; c < 4; ++c) {
                float r = qb[c];
                for (int i = 0; i < k; ++i) r = fmaf(t[i], E[i][c], r);
                d2 = fmaf(r, r, d2);
            }
            best = fminf(best, d2);
        } else {                                 // only the facets opposite negative weights
            for (int i = 0; i < k; ++i)
                if (t[i] < 0.0f) stack[sp++] = m & ~(1u << idx[i + 1]);
            if (wb < 0.0f) stack[sp++] = m & ~(1u << idx[0]);
        }
    }
    return best;
}

// All six Kuhn tetrahedra of the grid cell whose low corner is at integer offset (ox, oy, oz) from the reference
// voxel (3D grids).  d[S]: (D_e[c+S] - D_r[v]) / dD for the 8 corners S (bit0 = +x, bit1 = +y, bit2 = +z).
__device__ inline float ju_cell_min(const float (&d)[8], const GridP& g, int ox, int oy, int oz, float best2)
{
    const int perms[6][3] = {{1, 2, 4}, {1, 4, 2}, {2, 1, 4}, {2, 4, 1}, {4, 1, 2}, {4, 2, 1}};
    const float base[3] = {(float)ox * g.h[0], (float)oy * g.h[1], (float)oz * g.h[2]};
#pragma unroll 1
    for (int p = 0; p < 6; ++p) {
        float q[4][4];
        int S = 0;
        for (int v = 0; v < 4; ++v) {
            if (v > 0) S |= perms[p][v - 1];
            q[v][0] = base[0] + ((S & 1) ? g.h[0] : 0.0f);
            q[v][1] = base[1] + ((S & 2) ? g.h[1] : 0.0f);
            q[v][2] = base[2] + ((S & 4) ? g.h[2] : 0.0f);
            q[v][3] = d[S];
        }
        best2 = fminf(best2, ju_simplex_dist2(q, 0xFu));
    }
    return best2;
}

}  // namespace gamma_b200
