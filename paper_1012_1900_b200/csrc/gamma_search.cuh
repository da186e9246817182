// gamma_search.cuh -- subsystems (2) and (4): the gamma kernels.
//
//   k_max_ref       a0: D_norm = max(ref)                                   (reading 8)
//   k_prep_star     a1 + first part of a4: per voxel DD, cutoff, key (Algorithm A2 step 2 / CUDA Kernel 1,
//                   PAPER.md:231-233), block-local compaction of the evaluated voxels, then for interior
//                   voxels the 75 faces of the evaluation surface that touch the voxel ("star").  A voxel
//                   whose gamma_star is not larger than the distance to the rest of the surface is final;
//                   the others are appended to the search work list with key gamma_star (a much tighter
//                   key than |DD|/dD).
//   k_table_search  a4 + a5: Algorithm A1 step 4-b over the sorted offset table, G lanes
//                   cooperating on one reference voxel, running best shared by shuffles, exit when the
//                   table's L reaches the running gamma (reading 3); writes gamma at the voxel's own
//                   position (replaces the sort-back of A2 step 7).
// The point-to-simplex arithmetic is in features_generated.cuh.
#pragma once
#include "common.cuh"
#include "features_generated.cuh"

namespace gamma_b200 {

// ------------------------------------------------------------------------------------------------
// a0: max(ref)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_max_ref(const float* __restrict__ ref, int N, Ctl* __restrict__ ctl)
{
    float m = -INFINITY;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    if ((reinterpret_cast<uintptr_t>(ref) & 15u) == 0) {
        const float4* r4 = reinterpret_cast<const float4*>(ref);
        const int n4 = N >> 2;
        for (int i = tid; i < n4; i += nth) {
            const float4 v = __ldg(r4 + i);
            m = fmaxf(fmaxf(m, v.x), fmaxf(v.y, fmaxf(v.z, v.w)));
        }
        for (int i = (n4 << 2) + tid; i < N; i += nth) m = fmaxf(m, __ldg(ref + i));
    } else {
        for (int i = tid; i < N; i += nth) m = fmaxf(m, __ldg(ref + i));
    }
    m = warp_max(m);
    __shared__ float sm[8];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = threadIdx.x < 8 ? sm[threadIdx.x] : -INFINITY;
        m = warp_max(m);
        if (threadIdx.x == 0) atomicMax(&ctl->normOrd, float_to_ordered(m));
    }
}

// ------------------------------------------------------------------------------------------------
// a1 + star phase
// ------------------------------------------------------------------------------------------------
constexpr int PREP_THREADS = 256;
constexpr int PREP_TILE = 2048;

__device__ __forceinline__ float criterion_inv_dD(const EvalP& e, double dnorm, float Dr)
{
    const double dD = e.mode == 0 ? (double)e.DD * dnorm : (double)e.DD * (double)Dr;
    return dD > 0.0 ? (float)(1.0 / dD) : 0.0f;   // 0 marks "excluded: dD_v <= 0"
}

template <bool STAR>
__global__ void __launch_bounds__(PREP_THREADS)
k_prep_star(const float* __restrict__ ref, const float* __restrict__ ev, float* __restrict__ out, GridP g,
            EvalP e, Ctl* __restrict__ ctl, unsigned* __restrict__ listKey, unsigned* __restrict__ listIdx)
{
    __shared__ int sList[PREP_TILE];
    __shared__ unsigned sCnt;
    __shared__ float sMax[PREP_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31;
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const double thr = (double)e.cutoff * dnorm;      // decided in double (include/gamma_b200.h)
    const float invGlobal = criterion_inv_dD(e, dnorm, 0.0f);
    float maxKey = 0.0f;
    unsigned nEvalLocal = 0;
    const float qnan = __int_as_float(0x7fc00000);
    const int numTiles = (g.N + PREP_TILE - 1) / PREP_TILE;

    for (int tile = blockIdx.x; tile < numTiles; tile += gridDim.x) {
        if (tid == 0) sCnt = 0;
        __syncthreads();
        // ---- a1: exclusion + block-local compaction (keeps warps full for the arithmetic below)
#pragma unroll
        for (int j = 0; j < PREP_TILE / PREP_THREADS; ++j) {
            const int lin = tile * PREP_TILE + j * PREP_THREADS + tid;
            bool keep = false;
            if (lin < g.N) {
                const float Dr = __ldg(ref + lin);
                const bool excluded = ((double)Dr < thr) ||
                                      (e.mode == 0 ? !(invGlobal > 0.0f) : !((double)e.DD * (double)Dr > 0.0));
                if (excluded) out[lin] = qnan;
                keep = !excluded;
            }
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            unsigned base = 0;
            if (lane == 0 && bal) base = atomicAdd(&sCnt, (unsigned)__popc(bal));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (keep) sList[base + __popc(bal & ((1u << lane) - 1u))] = lin;
        }
        __syncthreads();
        const int cnt = (int)sCnt;
        if (tid == 0) nEvalLocal += cnt;
        // ---- star phase over the compacted voxels of this tile
        for (int j0 = 0; j0 < cnt; j0 += PREP_THREADS) {
            const int j = j0 + tid;
            bool toSearch = false;
            float key = 0.0f;
            int lin = 0;
            if (j < cnt) {
                lin = sList[j];
                const float Dr = __ldg(ref + lin);
                const float invdD = e.mode == 0 ? invGlobal : criterion_inv_dD(e, dnorm, Dr);
                const float d0 = (__ldg(ev + lin) - Dr) * invdD;
                key = fabsf(d0);                              // A1 step 4-a: gamma <- |DD| / dD
                toSearch = true;
                if (STAR && g.all_active) {
                    const int ix = lin % g.n[0], iy = (lin / g.n[0]) % g.n[1], iz = lin / g.stride[2];
                    const bool interior = ix >= 1 && ix <= g.n[0] - 2 && iy >= 1 && iy <= g.n[1] - 2 &&
                                          iz >= 1 && iz <= g.n[2] - 2;
                    if (interior) {
                        float d[27];
                        const float* p = ev + lin;
#pragma unroll
                        for (int oz = -1; oz <= 1; ++oz)
#pragma unroll
                            for (int oy = -1; oy <= 1; ++oy)
#pragma unroll
                                for (int ox = -1; ox <= 1; ++ox)
                                    d[(ox + 1) + 3 * (oy + 1) + 9 * (oz + 1)] =
                                        (__ldg(p + ox + oy * g.stride[1] + oz * g.stride[2]) - Dr) * invdD;
                        d[13] = d0;
                        const float gmax = gamma_star_gmax(d, g.invA);
                        key = key / sqrtf(gmax);              // gamma_star
                        if (key * key <= g.rho_link2) {       // nothing outside the star can be closer
                            out[lin] = key;
                            toSearch = false;
                        }
                    }
                }
                if (!(key == key)) {                          // non-finite doses: no search, NaN out
                    out[lin] = qnan;
                    toSearch = false;
                }
            }
            // append to the global work list (warp-aggregated)
            const unsigned bal = __ballot_sync(0xffffffffu, toSearch);
            if (bal) {
                unsigned base = 0;
                if (lane == __ffs(bal) - 1) base = atomicAdd(&ctl->nSearch, (unsigned)__popc(bal));
                base = __shfl_sync(0xffffffffu, base, __ffs(bal) - 1);
                if (toSearch) {
                    const unsigned pos = base + __popc(bal & ((1u << lane) - 1u));
                    listKey[pos] = __float_as_uint(key);
                    listIdx[pos] = (unsigned)lin;
                    maxKey = fmaxf(maxKey, key);
                }
            }
        }
        __syncthreads();
    }
    maxKey = warp_max(maxKey);
    if (lane == 0) sMax[tid >> 5] = maxKey;
    __syncthreads();
    if (tid == 0) {
        float m = 0.0f;
#pragma unroll
        for (int w = 0; w < PREP_THREADS / 32; ++w) m = fmaxf(m, sMax[w]);
        if (m > 0.0f) atomicMax(&ctl->maxKeyBits, __float_as_uint(m));
        if (nEvalLocal) atomicAdd(&ctl->nEval, nEvalLocal);
    }
}

// ------------------------------------------------------------------------------------------------
// a4: table search
// ------------------------------------------------------------------------------------------------
struct VoxelCtx {
    int v[3];
    int lin;
    float Dr, invdD;
};

// All 26 faces owned by the grid vertex c = v + o; returns the new best^2.
__device__ __forceinline__ float eval_owner_vertex(const float* __restrict__ ev, const GridP& g, const VoxelCtx& vc,
                                                   int ox, int oy, int oz, float best2)
{
    const int cx = vc.v[0] + ox, cy = vc.v[1] + oy, cz = vc.v[2] + oz;
    if ((unsigned)cx >= (unsigned)g.n[0] || (unsigned)cy >= (unsigned)g.n[1] || (unsigned)cz >= (unsigned)g.n[2])
        return best2;                                          // vertex outside the grid (reading 11)
    const unsigned usable = (cx + 1 < g.n[0] ? 1u : 0u) | (cy + 1 < g.n[1] ? 2u : 0u) | (cz + 1 < g.n[2] ? 4u : 0u);
    const int sx = (usable & 1u) ? 1 : 0, sy = (usable & 2u) ? g.stride[1] : 0, sz = (usable & 4u) ? g.stride[2] : 0;
    const float* p = ev + (vc.lin + ox + oy * g.stride[1] + oz * g.stride[2]);
    float d[8];
#pragma unroll
    for (int S = 0; S < 8; ++S)
        d[S] = (__ldg(p + ((S & 1) ? sx : 0) + ((S & 2) ? sy : 0) + ((S & 4) ? sz : 0)) - vc.Dr) * vc.invdD;
    const float fx = (float)ox, fy = (float)oy, fz = (float)oz;
    const float px = fx * g.h[0], py = fy * g.h[1], pz = fz * g.h[2];
    const float q[3] = {px * px, py * py, pz * pz};
    const float bxh = fx * g.hh[0], byh = fy * g.hh[1], bzh = fz * g.hh[2];
    float lam[8];
    lam[0] = 0.0f;
    lam[1] = -fx; lam[2] = -fy; lam[4] = -fz;
    lam[3] = -(bxh + byh) * g.invA[3];
    lam[5] = -(bxh + bzh) * g.invA[5];
    lam[6] = -(byh + bzh) * g.invA[6];
    lam[7] = -(bxh + byh + bzh) * g.invA[7];
    const float dxy = fx - fy, dxz = fx - fz, dyz = fy - fz;
    float X[8];
    X[0] = X[1] = X[2] = X[4] = 0.0f;
    X[3] = g.K3 * dxy * dxy;
    X[5] = g.K5 * dxz * dxz;
    X[6] = g.K6 * dyz * dyz;
    X[7] = g.Kxy7 * dxy * dxy + g.Kyz7 * dyz * dyz + g.Kzx7 * dxz * dxz;
    return gamma_owned_min(d, g.invA, lam, q, X, usable, best2);
}

template <int G>
__device__ __forceinline__ float group_min(float v)
{
#pragma unroll
    for (int s = G / 2; s > 0; s >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}

constexpr int SEARCH_THREADS = 256;

// G lanes per reference voxel: 1 (thread per voxel), 8 or 32.
template <int G>
__global__ void __launch_bounds__(SEARCH_THREADS)
k_table_search(const float* __restrict__ ref, const float* __restrict__ ev, float* __restrict__ out, GridP g,
               EvalP e, Ctl* __restrict__ ctl, const unsigned* __restrict__ listKey,
               const unsigned* __restrict__ listIdx, const int4* __restrict__ table)
{
    constexpr int VPW = 32 / G;                 // voxels per warp
    constexpr int EPP = G >= 8 ? G / 8 : 1;     // table entries per pass
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int gid = lane / G, gl = lane % G;
    const unsigned nS = ctl->nSearch, T = ctl->tableCount;
    const bool trunc = ctl->tableTrunc != 0;
    const float Rtab2 = ctl->Rtab2;
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const float invGlobal = criterion_inv_dD(e, dnorm, 0.0f);
    unsigned visits = 0;

    for (;;) {
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(&ctl->workCounter, (unsigned)VPW);
        base = __shfl_sync(FULL, base, 0);
        if (base >= nS) break;
        const unsigned item = base + gid;
        const bool have = item < nS;
        VoxelCtx vc;
        float key = 0.0f, best2 = 0.0f;
        if (have) {
            const unsigned idx = nS - 1u - item;              // deepest searches first
            vc.lin = (int)listIdx[idx];
            key = __uint_as_float(listKey[idx]);
            vc.Dr = __ldg(ref + vc.lin);
            vc.invdD = e.mode == 0 ? invGlobal : criterion_inv_dD(e, dnorm, vc.Dr);
            vc.v[0] = vc.lin % g.n[0];
            vc.v[1] = (vc.lin / g.n[0]) % g.n[1];
            vc.v[2] = vc.lin / g.stride[2];
            best2 = key * key;
        } else {
            vc.lin = 0; vc.Dr = 0.0f; vc.invdD = 0.0f; vc.v[0] = vc.v[1] = vc.v[2] = 0;
        }
        // ---- Algorithm A1 step 4-b over the sorted table
        for (unsigned e0 = 0;; e0 += EPP) {
            bool more = have && e0 < T;
            if (more) more = __int_as_float(__ldg(&table[e0].x)) < best2;    // 4-b-ii: stop at L >= gamma
            if (!__any_sync(FULL, more)) break;
            if (G >= 8) {
                const unsigned en = e0 + (unsigned)(gl >> 3);
                float cand = best2;
                if (more && en < T) {
                    const int4 t = __ldg(&table[en]);
                    if (__int_as_float(t.x) < best2) {
                        const int ox = (gl & 1) ? -t.y - 1 : t.y;
                        const int oy = (gl & 2) ? -t.z - 1 : t.z;
                        const int oz = (gl & 4) ? -t.w - 1 : t.w;
                        cand = eval_owner_vertex(ev, g, vc, ox, oy, oz, best2);
                        ++visits;
                    }
                }
                best2 = group_min<(G >= 8 ? G : 8)>(cand);
            } else {
                if (more) {
                    const int4 t = __ldg(&table[e0]);
#pragma unroll 1
                    for (int var = 0; var < 8; ++var) {
                        const int ox = (var & 1) ? -t.y - 1 : t.y;
                        const int oy = (var & 2) ? -t.z - 1 : t.z;
                        const int oz = (var & 4) ? -t.w - 1 : t.w;
                        best2 = eval_owner_vertex(ev, g, vc, ox, oy, oz, best2);
                        ++visits;
                    }
                }
            }
        }
        // ---- beyond a truncated table: exhaustive enumeration of the remaining octant box (exact, slow)
        if (trunc) {
            int rx = 0, ry = 0, rz = 0;
            unsigned V = 0;
            if (have && best2 > Rtab2) {
                const float b = sqrtf(best2);
                rx = g.h[0] > 0.0f ? (int)fminf((float)(g.n[0] - 1), floorf(b / g.h[0])) + 1 : 1;
                ry = g.h[1] > 0.0f ? (int)fminf((float)(g.n[1] - 1), floorf(b / g.h[1])) + 1 : 1;
                rz = g.h[2] > 0.0f ? (int)fminf((float)(g.n[2] - 1), floorf(b / g.h[2])) + 1 : 1;
                V = (unsigned)(rx * ry * rz);
            }
            for (unsigned i0 = 0;; i0 += EPP) {
                const bool more = i0 < V && best2 > Rtab2;
                if (!__any_sync(FULL, more)) break;
                if (G >= 8) {
                    const unsigned i = i0 + (unsigned)(gl >> 3);
                    float cand = best2;
                    if (more && i < V) {
                        const int mx = i % rx, my = (i / rx) % ry, mz = i / (rx * ry);
                        const float L2 = cell_L2(mx, my, mz, g);
                        if (L2 >= Rtab2 && L2 < best2) {
                            const int ox = (gl & 1) ? -mx - 1 : mx;
                            const int oy = (gl & 2) ? -my - 1 : my;
                            const int oz = (gl & 4) ? -mz - 1 : mz;
                            cand = eval_owner_vertex(ev, g, vc, ox, oy, oz, best2);
                            ++visits;
                        }
                    }
                    best2 = group_min<(G >= 8 ? G : 8)>(cand);
                } else if (more) {
                    const int mx = i0 % rx, my = (i0 / rx) % ry, mz = i0 / (rx * ry);
                    const float L2 = cell_L2(mx, my, mz, g);
                    if (L2 >= Rtab2 && L2 < best2) {
#pragma unroll 1
                        for (int var = 0; var < 8; ++var) {
                            const int ox = (var & 1) ? -mx - 1 : mx;
                            const int oy = (var & 2) ? -my - 1 : my;
                            const int oz = (var & 4) ? -mz - 1 : mz;
                            best2 = eval_owner_vertex(ev, g, vc, ox, oy, oz, best2);
                            ++visits;
                        }
                    }
                }
            }
        }
        if (have && gl == 0) out[vc.lin] = fminf(key, sqrtf(best2));   // a5: write at the voxel's own place
    }
    // diagnostic counter: one atomic per warp
    for (int s = 16; s > 0; s >>= 1) visits += __shfl_xor_sync(FULL, visits, s);
    if (lane == 0 && visits) atomicAdd(&ctl->visits, (unsigned long long)visits);
}

}  // namespace gamma_b200
