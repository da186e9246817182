// tile_star.cuh -- a1 + a2 + first part of a4 in ONE kernel over spatial tiles (BASELINE.json north_star (4):
// "evaluation-dose tiles plus halo staged by TMA into shared memory").
//
//   k_tile_star  a block owns a tile of 8 x 4 x 4 voxels at a time (one voxel per thread).  The evaluation doses of
//                the tile plus a halo of one voxel (a box of 16 x 6 x 6 floats that starts 4 voxels before the tile in x,
//                10 of the 16 used: the TMA wants the innermost start coordinate and the row length in multiples of
//                16 bytes -- an unaligned start is an illegal instruction on sm_100a, measured) and the reference doses
//                of the tile (8 x 4 x 4) are fetched by the TMA
//                (cp.async.bulk.tensor.3d, completion on an mbarrier, out-of-grid elements filled with zeros) into a
//                two-stage ring: while a tile is worked on, the next one is in flight.  Per tile: the cutoff decision
//                (k_classify's), NaN for excluded voxels, compaction of the evaluated voxels of the tile in shared
//                memory (so that the arithmetic runs on full warps where the tile is full), then the star phase of
//                k_star with the 27 doses read from shared memory, and the same two depth-class work lists appended.
//                No list of evaluated voxels is written or read, and k_classify is not launched: 3 kernels per call.
//
// LOADS: template parameter TMA = false is the same kernel with the tile filled by cooperative guarded loads (any nx,
// any alignment; also the B side of the A/B measurement in profiles/).  The TMA needs nx % 4 == 0 (global strides are
// multiples of 16 bytes) and 16-byte aligned ref / eval.
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "features_generated.cuh"
#include "offset_table.cuh"
#include "stats.cuh"

namespace gamma_b200 {

constexpr int TILE_X = 8, TILE_Y = 4, TILE_Z = 4;
constexpr int TILE_VOX = TILE_X * TILE_Y * TILE_Z;            // 128 = threads per block
constexpr int HALO_PX = 16, HALO_X0 = 4;                      // row of 16 floats starting at x0 - 4 (16-byte aligned start)
constexpr int HALO_Y = TILE_Y + 2, HALO_Z = TILE_Z + 2;
constexpr int HALO_ELEMS = HALO_PX * HALO_Y * HALO_Z;         // 576
constexpr int TILE_STAGES = 2;
constexpr unsigned TILE_TX_BYTES = (HALO_ELEMS + TILE_VOX) * 4;

struct TileSmem {
    alignas(128) float ev[TILE_STAGES][HALO_ELEMS];           // 2304 B per stage: every stage stays 128-byte aligned
    alignas(128) float ref[TILE_STAGES][TILE_VOX];
    alignas(8) unsigned long long bar[TILE_STAGES];
    unsigned char list[TILE_VOX];
    unsigned warpCnt[TILE_VOX / 32];
    int nextTile;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tile_barrier_init(unsigned long long* bar)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tile_barrier_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "TILE_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra TILE_DONE;\n"
        "bra TILE_WAIT;\n"
        "TILE_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// one thread: arm the barrier with the bytes of both boxes, then start the two tensor copies
__device__ __forceinline__ void tile_issue_tma(const CUtensorMap* mapRef, const CUtensorMap* mapEv, float* dstRef,
                                               float* dstEv, unsigned long long* bar, int x0, int y0, int z0)
{
    const unsigned b = smem_u32(bar);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(TILE_TX_BYTES) : "memory");
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dstEv)),
        "l"(mapEv), "r"(x0 - HALO_X0), "r"(y0 - 1), "r"(z0 - 1), "r"(b)
        : "memory");
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dstRef)),
        "l"(mapRef), "r"(x0), "r"(y0), "r"(z0), "r"(b)
        : "memory");
}

struct TileGrid {
    int tx, ty, tz;           // tiles per axis
    unsigned divMul[2], divSh[2];   // exact division by tx (0) and tx * ty (1): fast_div
};

#ifndef GAMMA_TILE_MIN_BLOCKS
#define GAMMA_TILE_MIN_BLOCKS 9
#endif

template <bool TMA>
__global__ void __launch_bounds__(TILE_VOX, GAMMA_TILE_MIN_BLOCKS)
k_tile_star(const __grid_constant__ CUtensorMap mapRef, const __grid_constant__ CUtensorMap mapEv,
            const float* __restrict__ ref, const float* __restrict__ ev, float* __restrict__ out, GridP g, EvalP e,
            Ctl* __restrict__ ctl, unsigned* __restrict__ listKey, unsigned* __restrict__ listIdx,
            unsigned* __restrict__ deepKey, unsigned* __restrict__ deepIdx, int buildTable,
            const __grid_constant__ TablePlan tabPlan, int4* __restrict__ table, unsigned* __restrict__ tmpL,
            unsigned* __restrict__ tmpIdx, StatsP st, TileGrid tg)
{
    using TabS = TableSmem<TAB_EMBED_ENTRIES, TAB_EMBED_BUCKETS, TAB_EMBED_BLOCKS>;
    using StatS = FusedStats<TILE_VOX>;
    __shared__ __align__(16) unsigned char sRaw[sizeof(TabS) > sizeof(StatS) ? sizeof(TabS) : sizeof(StatS)];
    __shared__ TileSmem T;
    __shared__ float sMax[TILE_VOX / 32];
    __shared__ unsigned sNan;
    StatS& sStat = *reinterpret_cast<StatS*>(sRaw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned FULL = 0xffffffffu;
    trace_first(e.call, 2);
    pdl_launch_dependents();
    const int numTiles = tg.tx * tg.ty * tg.tz;
    const int lx = tid & (TILE_X - 1), ly = (tid >> 3) & (TILE_Y - 1), lz = tid >> 5;
    auto tile_origin = [&](int t, int& x0, int& y0, int& z0) {
        const int tz = (int)fast_div((unsigned)t, tg.divMul[1], tg.divSh[1]);
        const int rem = t - tz * tg.tx * tg.ty;
        const int ty = (int)fast_div((unsigned)rem, tg.divMul[0], tg.divSh[0]);
        x0 = (rem - ty * tg.tx) * TILE_X; y0 = ty * TILE_Y; z0 = tz * TILE_Z;
    };
    // fill stage s with tile t: TMA (one thread, asynchronous) or cooperative guarded loads (all threads, synchronous
    // up to the barrier the caller places)
    auto fetch = [&](int t, int s) {
        int x0, y0, z0;
        tile_origin(t, x0, y0, z0);
        if (TMA) {
            if (tid == 0) tile_issue_tma(&mapRef, &mapEv, T.ref[s], T.ev[s], &T.bar[s], x0, y0, z0);
        } else {
            constexpr int USED_X = TILE_X + 2;            // the 10 columns of each 16-float row that are read
            for (int i = tid; i < USED_X * HALO_Y * HALO_Z; i += TILE_VOX) {
                const int hz = i / (USED_X * HALO_Y), r = i - hz * (USED_X * HALO_Y), hy = r / USED_X;
                const int hx = r - hy * USED_X + HALO_X0 - 1;
                const int gx = x0 - HALO_X0 + hx, gy = y0 - 1 + hy, gz = z0 - 1 + hz;
                const bool in = (unsigned)gx < (unsigned)g.n[0] && (unsigned)gy < (unsigned)g.n[1] && (unsigned)gz < (unsigned)g.n[2];
                T.ev[s][(hz * HALO_Y + hy) * HALO_PX + hx] = in ? __ldg(ev + (gx + gy * g.stride[1] + gz * g.stride[2])) : 0.0f;
            }
            const int gx = x0 + lx, gy = y0 + ly, gz = z0 + lz;
            const bool in = gx < g.n[0] && gy < g.n[1] && gz < g.n[2];
            T.ref[s][tid] = in ? __ldg(ref + (gx + gy * g.stride[1] + gz * g.stride[2])) : 0.0f;
        }
    };
    int tile = blockIdx.x;
    if (TMA) {
        if (tid == 0) {
            tile_barrier_init(&T.bar[0]);
            tile_barrier_init(&T.bar[1]);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncthreads();
        // ref / eval are inputs of the call (k_norm released this kernel only after their producer had completed):
        // the first tile is in flight while the table is built and k_norm drains
        if (tile < numTiles) fetch(tile, 0);
    }
    if (tid == 0) sNan = 0;
    // a3 inside the wait (as in k_star): the first blocks build the prefix table
    if (buildTable) {
        TabS& sTab = *reinterpret_cast<TabS*>(sRaw);
        for (int slice = blockIdx.x; slice < TAB_EMBED_BLOCKS; slice += gridDim.x)
            table_build_slice<TILE_VOX, TAB_EMBED_ENTRIES, TAB_EMBED_BUCKETS, TAB_EMBED_BLOCKS>(
                sTab, g, e, ctl, &tabPlan, 0.0f, TAB_EMBED_MAX_CELLS, table, tmpL, tmpIdx, slice);
    }
    pdl_wait();                                           // k_norm's maxima from here on
    trace_waited(e.call, 2);
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const double thr = (double)e.cutoff * dnorm;          // decided in double (include/gamma_b200.h)
    const float invGlobal = criterion_inv_dD(e, dnorm, 0.0f);
    const bool globalOk = invGlobal > 0.0f;
    if (blockIdx.x == 0 && tid == 0) ctl->invGlobal = invGlobal;          // k_table_search reads it from here
    const float qnan = __int_as_float(0x7fc00000);
    float A[8];
    A[0] = 0.0f;
#pragma unroll
    for (int S = 1; S < 8; ++S) A[S] = ((S & 1) ? g.hh[0] : 0.0f) + ((S & 2) ? g.hh[1] : 0.0f) + ((S & 4) ? g.hh[2] : 0.0f);
    float maxKey = 0.0f;
    unsigned nExcluded = 0, nNanKey = 0;
    fused_stats_init(sStat, st);
    __syncthreads();

    for (int it = 0; tile < numTiles; ++it) {
        const int s = it & 1;
        if (tid == 0) T.nextTile = (int)atomicAdd(&ctl->tileCounter, 1u) + (int)gridDim.x;
        if (!TMA) fetch(tile, s);
        __syncthreads();                                  // everyone has left the previous tile: its stage is free
        const int next = T.nextTile;
        if (TMA) {
            if (next < numTiles) fetch(next, s ^ 1);
            tile_barrier_wait(&T.bar[s], (unsigned)(it >> 1) & 1u);
        }
        int x0, y0, z0;
        tile_origin(tile, x0, y0, z0);
        // ---- a1: exclusion (k_classify's decision), NaN out, compaction of the tile's evaluated voxels
        const int gx = x0 + lx, gy = y0 + ly, gz = z0 + lz;
        const bool inGrid = gx < g.n[0] && gy < g.n[1] && gz < g.n[2];
        const int linMine = gx + gy * g.stride[1] + gz * g.stride[2];
        const float DrMine = T.ref[s][tid];
        const bool excluded = ((double)DrMine < thr) || (e.mode == 0 ? !globalOk : !((double)e.DD * (double)DrMine > 0.0));
        const bool keep = inGrid && !excluded;
        if (inGrid && excluded) { out[linMine] = qnan; ++nExcluded; }
        const unsigned bal = __ballot_sync(FULL, keep);
        if (lane == 0) T.warpCnt[warp] = (unsigned)__popc(bal);
        __syncthreads();
        unsigned before = 0, m = 0;
#pragma unroll
        for (int w = 0; w < TILE_VOX / 32; ++w) {
            const unsigned c = T.warpCnt[w];
            before += w < warp ? c : 0u;
            m += c;
        }
        if (m == 0) { tile = next; continue; }            // nothing to evaluate here (uniform over the block)
        if (keep) T.list[before + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)tid;
        if (tid == 0) atomicAdd(&ctl->nEval, m);
        __syncthreads();
        // ---- first part of a4: the star phase of k_star, doses from shared memory
        bool toSearch = false, starDone = false;
        float key = 0.0f;
        int lin = 0;
        if ((unsigned)tid < m) {
            const int v = (int)T.list[tid];
            const int vx = v & (TILE_X - 1), vy = (v >> 3) & (TILE_Y - 1), vz = v >> 5;
            const int ix = x0 + vx, iy = y0 + vy, iz = z0 + vz;
            lin = ix + iy * g.stride[1] + iz * g.stride[2];
            const float Dr = T.ref[s][v];
            const float invdD = e.mode == 0 ? invGlobal : criterion_inv_dD(e, dnorm, Dr);
            const float* p = &T.ev[s][((vz + 1) * HALO_Y + (vy + 1)) * HALO_PX + (vx + HALO_X0)];
            const float d0 = (p[0] - Dr) * invdD;
            key = fabsf(d0);                              // A1 step 4-a: gamma <- |DD| / dD
            toSearch = true;
            const bool interior = ix >= 1 && ix <= g.n[0] - 2 && iy >= 1 && iy <= g.n[1] - 2 && iz >= 1 && iz <= g.n[2] - 2;
            if (interior) {
                float d[27];
                float vb = d0 * d0;                       // squared distance to the nearest of the 27 grid points
                float dlo = d0, dhi = d0;                 // dose range of the 27 grid points
#pragma unroll
                for (int oz = -1; oz <= 1; ++oz)
#pragma unroll
                    for (int oy = -1; oy <= 1; ++oy)
#pragma unroll
                        for (int ox = -1; ox <= 1; ++ox) {
                            const int k = (ox + 1) + 3 * (oy + 1) + 9 * (oz + 1);
                            if (k == 13) { d[13] = d0; continue; }
                            const float dv = (p[ox + oy * HALO_PX + oz * HALO_PX * HALO_Y] - Dr) * invdD;
                            d[k] = dv;
                            vb = fminf(vb, fmaf(dv, dv, A[(ox ? 1 : 0) | (oy ? 2 : 0) | (oz ? 4 : 0)]));
                            dlo = fminf(dlo, dv);
                            dhi = fmaxf(dhi, dv);
                        }
                const float gmax = gamma_star_gmax(d, g.invA);
                starDone = true;
                key = key / sqrtf(gmax);                  // gamma_star
                const float dr = fmaxf(fmaxf(dlo, -dhi), 0.0f);
                const float outside2 = fminf(g.hmin2, fmaf(dr, dr, g.rho_link2));
                if (key * key <= outside2) {              // nothing outside the star can be closer (see k_star)
                    out[lin] = key;
                    fused_stats_add(sStat, st, key);
                    toSearch = false;
                } else {
                    key = fminf(key, sqrtf(vb));
                }
            }
            if (!(key == key)) {                          // non-finite doses: no search, NaN out
                out[lin] = qnan;
                ++nNanKey;
                toSearch = false;
            }
        }
        // ---- a2 as a 1-bit sort: ring items and deep items go to their own lists (warp-aggregated appends)
        const bool deep = toSearch && !(starDone && key * key < g.hmin2);
        const unsigned balR = __ballot_sync(FULL, toSearch && !deep);
        if (balR) {
            const int leader = __ffs(balR) - 1;
            unsigned base = 0;
            if (lane == leader) base = atomicAdd(&ctl->nSearch, (unsigned)__popc(balR));
            base = __shfl_sync(FULL, base, leader);
            if (toSearch && !deep) {
                const unsigned pos = base + __popc(balR & ((1u << lane) - 1u));
                listKey[pos] = __float_as_uint(key);
                listIdx[pos] = (unsigned)lin;
                maxKey = fmaxf(maxKey, key);
            }
        }
        const unsigned balD = __ballot_sync(FULL, deep);
        if (balD) {
            const int leader = __ffs(balD) - 1;
            unsigned base = 0;
            if (lane == leader) base = atomicAdd(&ctl->nDeep, (unsigned)__popc(balD));
            base = __shfl_sync(FULL, base, leader);
            if (deep) {
                const unsigned pos = base + __popc(balD & ((1u << lane) - 1u));
                deepKey[pos] = __float_as_uint(key);
                deepIdx[pos] = (unsigned)lin;
                maxKey = fmaxf(maxKey, key);
            }
        }
        tile = next;
    }
    maxKey = warp_max(maxKey);
    if (lane == 0) sMax[warp] = maxKey;
    if (st.hist) {
        nExcluded += nNanKey;
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) nExcluded += __shfl_xor_sync(FULL, nExcluded, sft);
        if (lane == 0 && nExcluded) atomicAdd(&sNan, nExcluded);
    }
    __syncthreads();
    if (tid == 0) {
        float mk = 0.0f;
#pragma unroll
        for (int w = 0; w < TILE_VOX / 32; ++w) mk = fmaxf(mk, sMax[w]);
        if (mk > 0.0f) atomicMax(&ctl->maxKeyBits, __float_as_uint(mk));
        if (st.hist && sNan) atomicAdd(&st.summary->n_nan, sNan);
    }
    fused_stats_flush(sStat, st);
    trace_last(e.call, 2);
}

}  // namespace gamma_b200
