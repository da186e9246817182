// general.cuh -- gamma_eval_general: the evaluation dose on ITS OWN grid (dims, spacing, origin), closest point of the
// evaluation surface as a second output (Eq. 1, does not need one grid; the
// refinements cited at PAPER.md:135 need the point where the minimum is attained).
//
// Same search as the same-grid path -- owner vertices visited in the order of the sorted offset table (Algorithm A1
// steps 2-4), the 26 owned faces of each by the closed form of features_generated.cuh, exit when the
// table's bound reaches the running gamma -- with two differences:
//   * the reference point is not an evaluation vertex, so there is no star / ring phase: every evaluated voxel walks
//     the table, 8 lanes per voxel (one octant of a table entry each), starting from the evaluation vertex c0 NEAREST
//     to the point.  With p = c0 + f (|f_a| <= 1/2 voxel inside the grid) the offset o of an owner vertex enters the
//     closed form as the real number o - f;
//   * the table is sorted by the bounds of a point AT a vertex.  For the displaced point every bound moves by at most
//     slack = |f o h| (triangle inequality), so the walk stops when L_table - slack >= gamma, and an owner vertex is
//     evaluated only if the EXACT minimum spatial distance of its cell to the point is below the running gamma.
// k_norm (max of ref) and k_classify (cutoff, NaN, compaction) are the same-grid kernels on the reference grid.
#pragma once
#include "common.cuh"
#include "features_generated.cuh"
#include "gamma_search.cuh"

namespace gamma_b200 {

struct GeneralP {
    int rn[3];                       // reference grid dims
    unsigned rDivMul[2], rDivSh[2];  // exact division by rn[0] and rn[0] * rn[1]
    double off[3], scale[3];         // evaluation index of reference voxel v: u_a = off_a + v_a * scale_a
    float eorg[3], esp[3];           // evaluation origin / spacing in mm (closest-point output)
};

constexpr int GENERAL_THREADS = 128;

// The 26 faces owned by evaluation vertex c = c0 + o against the point c0 + f; returns min(best2, ...).
__device__ __forceinline__ float general_owner_vertex(const float* __restrict__ ev, const GridP& g, const int (&c0)[3],
                                                      int lin0, const float (&f)[3], float Dr, float invdD, int ox, int oy,
                                                      int oz, float best2, bool wantLoc, float (&loc)[4],
                                                      float cellL2 = 0.0f, float prune2 = INFINITY)
{
    // cellL2: exact squared minimum spatial distance of the vertex's cell to the point; prune2: the running gamma^2 --
    // the vertex is skipped when nothing in its cell can be closer than that
    const int cx = c0[0] + ox, cy = c0[1] + oy, cz = c0[2] + oz;
    if ((unsigned)cx >= (unsigned)g.n[0] || (unsigned)cy >= (unsigned)g.n[1] || (unsigned)cz >= (unsigned)g.n[2])
        return best2;                                          // vertex outside the grid (reading 11)
    const unsigned usable = (cx + 1 < g.n[0] ? 1u : 0u) | (cy + 1 < g.n[1] ? 2u : 0u) | (cz + 1 < g.n[2] ? 4u : 0u);
    const int sx = (usable & 1u) ? 1 : 0, sy = (usable & 2u) ? g.stride[1] : 0, sz = (usable & 4u) ? g.stride[2] : 0;
    const float* p = ev + (lin0 + ox + oy * g.stride[1] + oz * g.stride[2]);
    float d[8];
#pragma unroll
    for (int S = 0; S < 8; ++S)
        d[S] = (__ldg(p + (((S & 1) ? sx : 0) + ((S & 2) ? sy : 0) + ((S & 4) ? sz : 0))) - Dr) * invdD;
    // exact prune: every face this vertex owns lies in its cell, whose points are at least cellL2 away
    // in space and carry a dose between the smallest and the largest of the eight corners
    {
        const float dlo = fminf(fminf(fminf(d[0], d[1]), fminf(d[2], d[3])), fminf(fminf(d[4], d[5]), fminf(d[6], d[7])));
        const float dhi = fmaxf(fmaxf(fmaxf(d[0], d[1]), fmaxf(d[2], d[3])), fmaxf(fmaxf(d[4], d[5]), fmaxf(d[6], d[7])));
        const float dr = fmaxf(fmaxf(dlo, -dhi), 0.0f);
        if (!(fmaf(dr, dr, cellL2) < prune2)) return best2;
    }
    float lam[8], q[3], X[8];
    owned_face_terms(g, (float)ox - f[0], (float)oy - f[1], (float)oz - f[2], usable, lam, q, X);
    if (wantLoc) return gamma_owned_argmin(d, g.invA, lam, q, X, usable, best2, loc);
    return gamma_owned_min(d, g.invA, lam, q, X, best2);
}

// exact squared minimum spatial distance (normalised) from the point c0 + f to the cell [c0 + o, c0 + o + 1]
__device__ __forceinline__ float general_cell_L2(const GridP& g, const float (&f)[3], int ox, int oy, int oz)
{
    const float ax = fmaxf(fmaxf((float)ox - f[0], f[0] - (float)(ox + 1)), 0.0f) * g.h[0];
    const float ay = fmaxf(fmaxf((float)oy - f[1], f[1] - (float)(oy + 1)), 0.0f) * g.h[1];
    const float az = fmaxf(fmaxf((float)oz - f[2], f[2] - (float)(oz + 1)), 0.0f) * g.h[2];
    return fmaf(ax, ax, fmaf(ay, ay, az * az));
}

__global__ void __launch_bounds__(GENERAL_THREADS)
k_general_search(const float* __restrict__ ref, const float* __restrict__ ev, float* __restrict__ out,
                 float4* __restrict__ closest, GridP g, GeneralP gp, EvalP e, Ctl* __restrict__ ctl,
                 const unsigned* __restrict__ evalIdx, const int4* __restrict__ table)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, gid = lane >> 3, gl = lane & 7;
    pdl_wait();                                          // k_classify's list, k_offset_table's table
    pdl_launch_dependents();
    const unsigned M = ctl->nEval;
    const unsigned T = ctl->tableCount;
    const bool trunc = ctl->tableTrunc != 0;
    const float Rtab2 = ctl->Rtab2;
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const float invGlobal = ctl->invGlobal;
    const unsigned numUnits = (M + 3u) / 4u;
    const unsigned warpsTotal = gridDim.x * (GENERAL_THREADS / 32);
    unsigned unit = blockIdx.x * (GENERAL_THREADS / 32) + (threadIdx.x >> 5);
    unsigned staticRounds = numUnits / warpsTotal;                // whole rounds are static, a small rest by tickets (k_star)
    const bool tickets = staticRounds && 2u * (numUnits - staticRounds * warpsTotal) < warpsTotal;
    if (!tickets) ++staticRounds;
    const unsigned one = ticket_one(ctl);
    unsigned round = 1;
    const float qnan = __int_as_float(0x7fc00000);
    while (unit < numUnits) {
        unsigned nextUnit = numUnits;
        if (round < staticRounds) nextUnit = unit + warpsTotal;
        else if (tickets && lane == 0) nextUnit = ticket_next(&ctl->workCounter, one) + staticRounds * warpsTotal;
        ++round;
        const unsigned item = unit * 4u + (unsigned)gid;
        const bool have = item < M;
        int c0[3] = {0, 0, 0}, lin0 = 0, linR = 0;
        float f[3] = {0.0f, 0.0f, 0.0f}, Dr = 0.0f, invdD = 0.0f, slack = 0.0f;
        if (have) {
            linR = (int)evalIdx[item];
            Dr = __ldg(ref + linR);
            invdD = e.mode == 0 ? invGlobal : criterion_inv_dD(e, dnorm, Dr);
            const int vz = (int)fast_div((unsigned)linR, gp.rDivMul[1], gp.rDivSh[1]);
            const int rem = linR - vz * gp.rn[0] * gp.rn[1];
            const int vy = (int)fast_div((unsigned)rem, gp.rDivMul[0], gp.rDivSh[0]);
            const int v[3] = {rem - vy * gp.rn[0], vy, vz};
            float s2 = 0.0f;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double u = fma((double)v[a], gp.scale[a], gp.off[a]);   // evaluation index of the reference point
                double c = rint(u);
                c = fmin(fmax(c, 0.0), (double)(g.n[a] - 1));
                c0[a] = (int)c;
                f[a] = (float)(u - c);
                const float t = f[a] * g.h[a];
                s2 = fmaf(t, t, s2);
            }
            slack = sqrtf(s2) * 1.000001f;
            lin0 = c0[0] + c0[1] * g.stride[1] + c0[2] * g.stride[2];
        }
        float best2 = INFINITY;                          // gamma^2 so far (the first pass, offset 0, always finds a vertex)
        float mine2 = INFINITY;                          // best of the owner vertices THIS lane evaluated, and which one
        int mo[3] = {0, 0, 0};
        float loc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        auto visit = [&](int ox, int oy, int oz, float cellL2) -> float {
            const float own = general_owner_vertex(ev, g, c0, lin0, f, Dr, invdD, ox, oy, oz, INFINITY, false, loc, cellL2, best2);
            if (own < mine2) { mine2 = own; mo[0] = ox; mo[1] = oy; mo[2] = oz; }
            return fminf(best2, own);
        };
        // ---- Algorithm A1 step 4-b over the sorted table, one entry (8 octants) per pass
        for (unsigned en = 0;; ++en) {
            bool more = have && en < T;
            float Lt = 0.0f;
            if (more) {
                Lt = sqrtf(__int_as_float(__ldg(&table[en].x)));
                const float reach = fmaxf(Lt - slack, 0.0f);
                more = reach * reach < best2;            // 4-b-ii with the slack of the displaced point
            }
            if (!__any_sync(FULL, more)) break;
            float cand = best2;
            if (more) {
                const int4 t = __ldg(&table[en]);
                const int ox = (gl & 1) ? -t.y - 1 : t.y;
                const int oy = (gl & 2) ? -t.z - 1 : t.z;
                const int oz = (gl & 4) ? -t.w - 1 : t.w;
                const float cL2 = general_cell_L2(g, f, ox, oy, oz);
                if (cL2 < best2) cand = visit(ox, oy, oz, cL2);
            }
            best2 = group_min<8>(cand);
        }
        // ---- beyond a truncated (prefix) table: Chebyshev shells of octant cells (as in search_items), with the slack
        if (trunc) {
            const int shMax = max(g.n[0], max(g.n[1], g.n[2])) - 1;
            const float hmin = sqrtf(g.hmin2);
            for (int sh = 0; sh <= shMax; ++sh) {
                const float reach = fmaxf((float)sh * hmin - slack, 0.0f);
                const bool go = have && reach * reach < best2;
                if (!__any_sync(FULL, go)) break;
                const int ey = min(sh, g.n[1] - 1), ez = min(sh, g.n[2] - 1);
                const int exm = min(sh - 1, g.n[0] - 1), eym = min(sh - 1, g.n[1] - 1);
                const unsigned cX = sh <= g.n[0] - 1 ? (unsigned)((ey + 1) * (ez + 1)) : 0u;
                const unsigned cY = (sh >= 1 && sh <= g.n[1] - 1) ? (unsigned)((exm + 1) * (ez + 1)) : 0u;
                const unsigned cZ = (sh >= 1 && sh <= g.n[2] - 1) ? (unsigned)((exm + 1) * (eym + 1)) : 0u;
                const unsigned V = cX + cY + cZ;
                for (unsigned i = 0; i < V; ++i) {
                    float cand = best2;
                    if (go) {
                        int mx, my, mz;
                        if (i < cX) { mx = sh; my = (int)(i % (unsigned)(ey + 1)); mz = (int)(i / (unsigned)(ey + 1)); }
                        else if (i < cX + cY) { const unsigned j = i - cX; my = sh; mx = (int)(j % (unsigned)(exm + 1)); mz = (int)(j / (unsigned)(exm + 1)); }
                        else { const unsigned j = i - cX - cY; mz = sh; mx = (int)(j % (unsigned)(exm + 1)); my = (int)(j / (unsigned)(exm + 1)); }
                        if (cell_L2(mx, my, mz, g) >= Rtab2) {           // the table has not covered this entry
                            const int ox = (gl & 1) ? -mx - 1 : mx;
                            const int oy = (gl & 2) ? -my - 1 : my;
                            const int oz = (gl & 4) ? -mz - 1 : mz;
                            const float cL2 = general_cell_L2(g, f, ox, oy, oz);
                if (cL2 < best2) cand = visit(ox, oy, oz, cL2);
                        }
                    }
                    best2 = group_min<8>(cand);
                }
            }
        }
        // ---- a5 + closest point: the lane whose owner vertex gave the minimum evaluates it once more with the foot point
        const unsigned balWin = __ballot_sync(FULL, have && mine2 == best2);
        if (have) {
            const float gam = sqrtf(best2);
            const bool nan = !(gam == gam);
            if (gl == 0) out[linR] = nan ? qnan : gam;
            if (closest) {
                const unsigned winners = (balWin >> (gid * 8)) & 0xffu;
                const int wl = winners ? __ffs(winners) - 1 : 0;
                if (gl == wl) {
                    float4 cp = make_float4(qnan, qnan, qnan, qnan);
                    if (!nan && winners) {
                        general_owner_vertex(ev, g, c0, lin0, f, Dr, invdD, mo[0], mo[1], mo[2], INFINITY, true, loc);
                        cp.x = gp.eorg[0] + ((float)(c0[0] + mo[0]) + loc[0]) * gp.esp[0];
                        cp.y = gp.eorg[1] + ((float)(c0[1] + mo[1]) + loc[1]) * gp.esp[1];
                        cp.z = gp.eorg[2] + ((float)(c0[2] + mo[2]) + loc[2]) * gp.esp[2];
                        cp.w = fmaf(loc[3], 1.0f / invdD, Dr);
                    }
                    closest[linR] = cp;
                }
            }
        }
        unit = __shfl_sync(FULL, nextUnit, 0);
    }
}

}  // namespace gamma_b200
