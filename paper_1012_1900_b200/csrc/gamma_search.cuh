// gamma_search.cuh -- subsystems (2) and (4): the gamma kernels.
//
//   k_norm           a0 + A1 step 1: D_norm = max(ref) (reading 8) and max |D_r - D_e|,
//                    which bounds every key and so fixes the radius of the offset table before the search
//                    list exists; zeroes the caller's fused-statistics buffers and the control block of the NEXT call.
//   k_classify       a1: cutoff decision, NaN for excluded voxels, compaction of the evaluated voxels.
// Consecutive kernels of a call are chained by programmatic dependent launch (pdl_wait / pdl_launch_dependents).
//   k_star           a1 + first part of a4: per evaluated voxel (from k_classify's compacted list) DD and key
//                    (Algorithm A2 step 2 / CUDA Kernel 1), then interior voxels try the 75 faces of
//                    the evaluation surface that touch the voxel ("star").  A voxel whose gamma_star is not larger
//                    than the distance to the rest of the surface is final; the others are appended to the
//                    search work list with key gamma_star (a much tighter key than |DD|/dD),
//                    split into depth classes (presort 4) or counted into the digit histogram of the presort.
//   k_bucket_scatter a2: one-pass MSD radix presort of the work list on the 8-bit key digit.
//   k_table_search   a4 + a5: Algorithm A1 step 4-b over the sorted offset table, G lanes
//                    cooperating on one reference voxel, running best shared by shuffles, exit when the
//                    table's L reaches the running gamma (reading 3); writes gamma at the voxel's own
//                    position (replaces the sort-back of A2 step 7).
// The point-to-simplex arithmetic is in features_generated.cuh.
#pragma once
#include "common.cuh"
#include "features_generated.cuh"
#include "offset_table.cuh"
#include "ju_simplex.cuh"
#include "stats.cuh"

namespace gamma_b200 {

__device__ __forceinline__ float block_max_256(float v, float* sm8)
{
    v = warp_max(v);
    if ((threadIdx.x & 31) == 0) sm8[threadIdx.x >> 5] = v;
    __syncthreads();
    float m = sm8[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) m = fmaxf(m, sm8[w]);
    __syncthreads();
    return m;
}

// ------------------------------------------------------------------------------------------------
// a0 + A1 step 1: max(ref), max |ref - eval| (and max |ref - eval| / ref for the local criterion)
// ------------------------------------------------------------------------------------------------
constexpr int NORM_THREADS = 256;

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Programmatic dependent launch (sm_90+): a kernel launched with the programmatic-serialisation attribute may
// start while its predecessor in the stream drains; it must not touch the predecessor's results before pdl_wait().
// Both are no-ops for a kernel launched without the attribute.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }


__global__ void __launch_bounds__(NORM_THREADS)
k_norm(const float* __restrict__ ref, const float* __restrict__ ev, int N, int mode, Ctl* __restrict__ cur,
       Ctl* __restrict__ next, int waitFirst, unsigned call, StatsP st, int needDD)
{
    // needDD == 0: only max(ref) is wanted -- the default prefix table does not depend on max |DD| (A1 step 1 sizes the
    // PAPER's table, opts.table_radius = 2), so the evaluation dose is not read here at all: 4 instead of 8 bytes per voxel
    trace_first(call, 0);
    // waitFirst: ref / eval may be results of the operation in front of this call: nothing is read before that
    // operation has completed -- and the dependents (k_classify fetches ref before its own wait) are released only
    // after that.  Otherwise (library-owned stream, the operation in front is the previous call's k_table_search,
    // which triggers its dependents at once) this kernel runs in the tail of that call: it reads this call's inputs
    // only, writes control blocks that call does not use, and waits for its end as its LAST act, so that nothing
    // after it can overtake the previous call.
    if (waitFirst) pdl_wait();
    pdl_launch_dependents();
    trace_waited(call, 0);
    if (blockIdx.x == gridDim.x - 1 && next != nullptr) {      // the next call finds its control block cleared
        unsigned* w = reinterpret_cast<unsigned*>(next);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctl) / 4); i += NORM_THREADS) w[i] = 0u;
    }
    if (st.hist) {                                              // a6 fused: the caller's buffers start from zero
        for (int b = blockIdx.x * NORM_THREADS + threadIdx.x; b < st.nbins; b += gridDim.x * NORM_THREADS) st.hist[b] = 0ull;
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            gamma_summary z;
            z.n_eval = 0; z.n_pass = 0; z.sum_gamma = 0.0; z.sum_gamma3 = 0.0; z.max_gamma = 0.0f; z.n_nan = 0; z.pad_ = 0;
            *st.summary = z;
        }
    }
    float m = -INFINITY, a = 0.0f, r = 0.0f;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    auto one = [&](float Dr, float De) {
        m = fmaxf(m, Dr);
        const float ad = fabsf(Dr - De);
        a = fmaxf(a, ad);                                       // fmaxf drops NaN
        if (mode == 1 && Dr > 0.0f) r = fmaxf(r, ad / Dr);
    };
    if (!needDD) {
        if ((reinterpret_cast<uintptr_t>(ref) & 15u) == 0) {
            const float4* r4 = reinterpret_cast<const float4*>(ref);
            const int n4 = N >> 2;
            int i = tid;
            for (; i + 3 * nth < n4; i += 4 * nth) {         // 4 independent 16-byte loads in flight per thread
                const float4 x0 = __ldg(r4 + i), x1 = __ldg(r4 + i + nth), x2 = __ldg(r4 + i + 2 * nth), x3 = __ldg(r4 + i + 3 * nth);
                m = fmaxf(fmaxf(fmaxf(m, x0.x), fmaxf(x0.y, x0.z)), fmaxf(fmaxf(x0.w, x1.x), fmaxf(x1.y, x1.z)));
                m = fmaxf(fmaxf(fmaxf(m, x1.w), fmaxf(x2.x, x2.y)), fmaxf(fmaxf(x2.z, x2.w), fmaxf(x3.x, x3.y)));
                m = fmaxf(m, fmaxf(x3.z, x3.w));
            }
            for (; i < n4; i += nth) {
                const float4 x = __ldg(r4 + i);
                m = fmaxf(fmaxf(m, x.x), fmaxf(fmaxf(x.y, x.z), x.w));
            }
            for (int k = (n4 << 2) + tid; k < N; k += nth) m = fmaxf(m, __ldg(ref + k));
        } else {
            for (int i = tid; i < N; i += nth) m = fmaxf(m, __ldg(ref + i));
        }
    } else if (((reinterpret_cast<uintptr_t>(ref) | reinterpret_cast<uintptr_t>(ev)) & 15u) == 0) {
        const float4* r4 = reinterpret_cast<const float4*>(ref);
        const float4* e4 = reinterpret_cast<const float4*>(ev);
        const int n4 = N >> 2;
        int i = tid;
        for (; i + 3 * nth < n4; i += 4 * nth) {             // large grids: 8 independent 16-byte loads in flight per thread
            const float4 x0 = __ldg(r4 + i), y0 = __ldg(e4 + i), x1 = __ldg(r4 + i + nth), y1 = __ldg(e4 + i + nth);
            const float4 x2 = __ldg(r4 + i + 2 * nth), y2 = __ldg(e4 + i + 2 * nth);
            const float4 x3 = __ldg(r4 + i + 3 * nth), y3 = __ldg(e4 + i + 3 * nth);
            one(x0.x, y0.x); one(x0.y, y0.y); one(x0.z, y0.z); one(x0.w, y0.w);
            one(x1.x, y1.x); one(x1.y, y1.y); one(x1.z, y1.z); one(x1.w, y1.w);
            one(x2.x, y2.x); one(x2.y, y2.y); one(x2.z, y2.z); one(x2.w, y2.w);
            one(x3.x, y3.x); one(x3.y, y3.y); one(x3.z, y3.z); one(x3.w, y3.w);
        }
        for (; i < n4; i += nth) {
            const float4 x = __ldg(r4 + i), y = __ldg(e4 + i);
            one(x.x, y.x); one(x.y, y.y); one(x.z, y.z); one(x.w, y.w);
        }
        for (int i = (n4 << 2) + tid; i < N; i += nth) one(__ldg(ref + i), __ldg(ev + i));
    } else {
        for (int i = tid; i < N; i += nth) one(__ldg(ref + i), __ldg(ev + i));
    }
    __shared__ float sm8[8];
    m = block_max_256(m, sm8);
    a = block_max_256(a, sm8);
    if (mode == 1) r = block_max_256(r, sm8);
    if (threadIdx.x == 0) {
        atomicMax(&cur->normOrd, float_to_ordered(m));
        if (a > 0.0f) atomicMax(&cur->maxAbsDD, __float_as_uint(a));
        if (r > 0.0f) atomicMax(&cur->maxRatio, __float_as_uint(r));
        // started early: one block holds the grid open until the previous call has ended (the kernels after this one
        // reuse its work lists); the other blocks give their registers back at once
        if (!waitFirst && blockIdx.x == 0) pdl_wait();
    }
    trace_last(call, 0);
}

// ------------------------------------------------------------------------------------------------
// a1: exclusion + compaction of the evaluated voxels (Algorithm A2 step 2 / CUDA Kernel 1)
// A pure stream over ref: float4 in, NaN out for excluded voxels, indices of evaluated voxels appended to
// evalIdx in chunk order (so neighbours stay neighbours).  One global atomic per 1024-voxel chunk.
// ------------------------------------------------------------------------------------------------
constexpr int PREP_THREADS = 256;
constexpr int PREP_CHUNK = 4 * PREP_THREADS;

__device__ __forceinline__ float criterion_inv_dD(const EvalP& e, double dnorm, float Dr)
{
    const double dD = e.mode == 0 ? (double)e.DD * dnorm : (double)e.DD * (double)Dr;
    return dD > 0.0 ? (float)(1.0 / dD) : 0.0f;   // 0 marks "excluded: dD_v <= 0"
}

__global__ void __launch_bounds__(PREP_THREADS)
k_classify(const float* __restrict__ ref, float* __restrict__ out, GridP g, EvalP e, Ctl* __restrict__ ctl,
           unsigned* __restrict__ evalIdx, StatsP st, Ctl* __restrict__ next, int first)
{
    // first != 0: the call has no k_norm (opts.norm_dose given, prefix table, no fused statistics: nothing of a0 is
    // needed) and this is its first kernel -- it waits for the operation in front of it before it reads anything and
    // zeroes the control block of the next call (`next`) in k_norm's place
    __shared__ unsigned sWarp[PREP_THREADS / 32];
    __shared__ unsigned sBase;
    __shared__ unsigned sNan;
    unsigned nExcluded = 0;                           // a6 fused: excluded voxels of this thread
    if (threadIdx.x == 0) sNan = 0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned FULL = 0xffffffffu;
    const int numChunks = (g.N + PREP_CHUNK - 1) / PREP_CHUNK;
    const bool vec = ((reinterpret_cast<uintptr_t>(ref) | reinterpret_cast<uintptr_t>(out)) & 15u) == 0;
    auto load_chunk = [&](int chunk, float (&Dr)[4]) -> int {
        const int lin0 = chunk * PREP_CHUNK + tid * 4;
        int nval = 0;
        if (vec && lin0 + 3 < g.N) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(ref + lin0));
            Dr[0] = v.x; Dr[1] = v.y; Dr[2] = v.z; Dr[3] = v.w;
            nval = 4;
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (lin0 + j < g.N) { Dr[j] = __ldg(ref + lin0 + j); nval = j + 1; } else Dr[j] = 0.0f;
        }
        return nval;
    };
    if (first) pdl_wait();
    pdl_launch_dependents();
    trace_first(e.call, 1);
    if (next != nullptr && blockIdx.x == gridDim.x - 1) {
        unsigned* w = reinterpret_cast<unsigned*>(next);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctl) / 4); i += PREP_THREADS) w[i] = 0u;
    }
    // ref is an input of the call, not a result of k_norm: the first chunk is fetched while k_norm drains
    float Dr[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    int nval = 0;
    if ((int)blockIdx.x < numChunks) nval = load_chunk(blockIdx.x, Dr);
    pdl_wait();                                       // k_norm's maxima from here on
    trace_waited(e.call, 1);
    // The cutoff is decided in double (include/gamma_b200.h): D_r < cutoff * D_norm.  For a float D_r that is the same
    // as D_r < thrUp with thrUp = the product rounded UP to float (if the product is a float, thrUp is the product;
    // otherwise no float lies between it and thrUp) -- one fp32 compare per voxel, same decision bit for bit.  Likewise
    // DD * D_r > 0 in double <=> D_r > 0 (DD > 0; the product of two floats cannot underflow in double).
    // The two constants take a double-precision division: one thread per block computes them (every thread doing so
    // was 40 % of this kernel's instructions, a thread here has one chunk of four voxels).
    __shared__ float sThrUp, sInvGlobal;
    if (tid == 0) {
        const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
        const double dnorm = (double)dnormF;
        sThrUp = __double2float_ru((double)e.cutoff * dnorm);
        sInvGlobal = criterion_inv_dD(e, dnorm, 0.0f);
        if (blockIdx.x == 0) ctl->invGlobal = sInvGlobal;   // the later kernels read it from here
    }
    __syncthreads();
    const float thrUp = sThrUp;
    const float invGlobal = sInvGlobal;
    const bool globalOk = invGlobal > 0.0f;
    const float qnan = __int_as_float(0x7fc00000);

    for (int chunk = blockIdx.x; chunk < numChunks; chunk += gridDim.x) {
        const int lin0 = chunk * PREP_CHUNK + tid * 4;
        if (chunk != (int)blockIdx.x) nval = load_chunk(chunk, Dr);
        unsigned keepMask = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const bool excluded = (Dr[j] < thrUp) || (e.mode == 0 ? !globalOk : !(Dr[j] > 0.0f));
            if (j < nval && !excluded) keepMask |= 1u << j;
        }
        if (keepMask == 0 && nval == 4 && vec) {
            *reinterpret_cast<float4*>(out + lin0) = make_float4(qnan, qnan, qnan, qnan);
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (j < nval && !(keepMask & (1u << j))) out[lin0 + j] = qnan;
        }
        const int c = __popc(keepMask);
        nExcluded += (unsigned)(nval - c);
        int incl = c;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const int t = __shfl_up_sync(FULL, incl, s);
            if (lane >= s) incl += t;
        }
        if (lane == 31) sWarp[warp] = (unsigned)incl;
        __syncthreads();
        if (tid == 0) {
            unsigned tot = 0;
#pragma unroll
            for (int w = 0; w < PREP_THREADS / 32; ++w) { const unsigned t = sWarp[w]; sWarp[w] = tot; tot += t; }
            sBase = tot ? atomicAdd(&ctl->nEval, tot) : 0u;
        }
        __syncthreads();
        unsigned pos = sBase + sWarp[warp] + (unsigned)(incl - c);
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (keepMask & (1u << j)) evalIdx[pos++] = (unsigned)(lin0 + j);
        __syncthreads();
    }
    if (st.hist) {
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) nExcluded += __shfl_xor_sync(FULL, nExcluded, s);
        if (lane == 0 && nExcluded) atomicAdd(&sNan, nExcluded);
        __syncthreads();
        if (tid == 0 && sNan) atomicAdd(&st.summary->n_nan, sNan);
    }
    trace_last(e.call, 1);
}

// ------------------------------------------------------------------------------------------------
// first part of a4: the star phase over the compacted voxels, one voxel per thread, one warp per 32
// consecutive list entries (whole rounds static, the last partial round fetched dynamically).
// ------------------------------------------------------------------------------------------------
// 128 threads x 9 resident blocks = 36 warps per SM at 56 registers: 148 x 36 x 32 = 170 496 voxels are in flight at
// once, so cases up to that many evaluated voxels (cfg2, cfg3: 160 256) finish in ONE round of items.
#ifndef GAMMA_STAR_THREADS
#define GAMMA_STAR_THREADS 128
#endif
constexpr int STAR_THREADS = GAMMA_STAR_THREADS;
#ifndef GAMMA_STAR_MIN_BLOCKS
#define GAMMA_STAR_MIN_BLOCKS 9
#endif

template <bool STAR>
__global__ void __launch_bounds__(STAR_THREADS, GAMMA_STAR_MIN_BLOCKS)
k_star(const float* __restrict__ ref, const float* __restrict__ ev, float* __restrict__ out, GridP g, EvalP e,
       Ctl* __restrict__ ctl, const unsigned* __restrict__ evalIdx, unsigned* __restrict__ listKey,
       unsigned* __restrict__ listIdx, unsigned* __restrict__ deepKey, unsigned* __restrict__ deepIdx, int classes,
       int buildTable, const __grid_constant__ TablePlan tabPlan, int4* __restrict__ table,
       unsigned* __restrict__ tmpL, unsigned* __restrict__ tmpIdx, StatsP st)
{
    // classes != 0: the work list is split by depth class at append time instead of being sorted afterwards --
    // "deep" items (key beyond the first non-zero table distance: the walk will pass table entry 0) go to
    // (deepKey, deepIdx), the others to (listKey, listIdx); no digit histogram is kept.
    __shared__ unsigned sHist[KEY_DIGITS];
    __shared__ float sMax[STAR_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned FULL = 0xffffffffu;
    pdl_launch_dependents();
    trace_first(e.call, 2);
    for (int d = tid; d < KEY_DIGITS; d += STAR_THREADS) sHist[d] = 0;
    // a3 inside the wait: the prefix table depends on the geometry only, so the first blocks build it (one slice of
    // buckets each) while k_classify is still running -- no side stream, no join, nothing added to the chain.
    // the table builder's working set and the fused-statistics slots share one piece of shared memory: the table is
    // finished (table_build_slice ends with a barrier) before the first voxel is looked at
    using TabS = TableSmem<TAB_EMBED_ENTRIES, TAB_EMBED_BUCKETS, TAB_EMBED_BLOCKS>;
    using StatS = FusedStats<STAR_THREADS>;
    __shared__ __align__(16) unsigned char sRaw[sizeof(TabS) > sizeof(StatS) ? sizeof(TabS) : sizeof(StatS)];
    StatS& sStat = *reinterpret_cast<StatS*>(sRaw);
    if (buildTable) {
        TabS& sTab = *reinterpret_cast<TabS*>(sRaw);
        for (int slice = blockIdx.x; slice < TAB_EMBED_BLOCKS; slice += gridDim.x)
            table_build_slice<STAR_THREADS, TAB_EMBED_ENTRIES, TAB_EMBED_BUCKETS, TAB_EMBED_BLOCKS>(
                sTab, g, e, ctl, &tabPlan, 0.0f, TAB_EMBED_MAX_CELLS, table, tmpL, tmpIdx, slice);
    }
    pdl_wait();                                           // k_classify's results from here on
    trace_waited(e.call, 2);
    // The index of the warp's first voxel is fetched together with the control block, not after it: one L2 round
    // trip less in front of the first round.  Entries at or beyond M are never used (and never dereferenced).
    unsigned item = blockIdx.x * (STAR_THREADS / 32) + (tid >> 5);
    unsigned linAhead = item * 32u + lane < (unsigned)g.N ? evalIdx[item * 32u + lane] : 0u;
    const unsigned M = ctl->nEval;
    const unsigned warpsTotal = gridDim.x * (STAR_THREADS / 32);
    const unsigned numItems = (M + 31u) / 32u;
    // Items are handed out in static rounds (item = warp + round * warps) while whole rounds are left; only a last,
    // partial round of less than half the warps goes through the ticket counter: 5 000 warps asking one address for a ticket at the same moment
    // queue up for microseconds (same-address atomics are served one at a time).
    unsigned staticRounds = numItems / warpsTotal;
    const bool tickets = staticRounds && 2u * (numItems - staticRounds * warpsTotal) < warpsTotal;
    if (!tickets) ++staticRounds;                          // a last round of half the warps or more is static too
    const unsigned one = ticket_one(ctl);
    unsigned round = 1;
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const float invGlobal = ctl->invGlobal;
    const float qnan = __int_as_float(0x7fc00000);
    // squared spatial distance of the 26 neighbours, by the set T of axes they differ in
    float A[8];
    A[0] = 0.0f;
#pragma unroll
    for (int T = 1; T < 8; ++T) A[T] = ((T & 1) ? g.hh[0] : 0.0f) + ((T & 2) ? g.hh[1] : 0.0f) + ((T & 4) ? g.hh[2] : 0.0f);
    float maxKey = 0.0f;
    fused_stats_init(sStat, st);
    unsigned nNanKey = 0;
    __syncthreads();

    while (item < numItems) {
        unsigned nextItem = numItems;
        if (round < staticRounds) nextItem = item + warpsTotal;
        else if (tickets && lane == 0) nextItem = ticket_next(&ctl->tileCounter, one) + staticRounds * warpsTotal;
        ++round;
        const unsigned j = item * 32u + lane;
        bool toSearch = false, starDone = false;
        float key = 0.0f;
        int lin = 0;
        if (j < M) {
            lin = (int)linAhead;
            const float Dr = __ldg(ref + lin);
            const float invdD = e.mode == 0 ? invGlobal : criterion_inv_dD(e, dnorm, Dr);
            const float d0 = (__ldg(ev + lin) - Dr) * invdD;
            key = fabsf(d0);                              // A1 step 4-a: gamma <- |DD| / dD
            toSearch = true;
            if (STAR && g.all_active) {
                int ix, iy, iz;
                voxel_coords(g, lin, ix, iy, iz);
                const bool interior = ix >= 1 && ix <= g.n[0] - 2 && iy >= 1 && iy <= g.n[1] - 2 &&
                                      iz >= 1 && iz <= g.n[2] - 2;
                if (interior) {
                    float d[27];
                    const float* p = ev + lin;
                    float vb = d0 * d0;                   // squared distance to the nearest of the 27 grid points
                    float dlo = d0, dhi = d0;             // dose range of the 27 grid points
#pragma unroll
                    for (int oz = -1; oz <= 1; ++oz)
#pragma unroll
                        for (int oy = -1; oy <= 1; ++oy)
#pragma unroll
                            for (int ox = -1; ox <= 1; ++ox) {
                                const int k = (ox + 1) + 3 * (oy + 1) + 9 * (oz + 1);
                                if (k == 13) { d[13] = d0; continue; }
                                const float dv = (__ldg(p + ox + oy * g.stride[1] + oz * g.stride[2]) - Dr) * invdD;
                                d[k] = dv;
                                vb = fminf(vb, fmaf(dv, dv, A[(ox ? 1 : 0) | (oy ? 2 : 0) | (oz ? 4 : 0)]));
                                dlo = fminf(dlo, dv);
                                dhi = fmaxf(dhi, dv);
                            }
                    const float gmax = gamma_star_gmax(d, g.invA);
                    starDone = true;
                    key = key / sqrtf(gmax);              // gamma_star
                    // Lower bound of everything OUTSIDE the star: beyond the 8 touching cells the spatial distance
                    // alone is >= hmin; inside them (but outside the star) it is >= rho_link and the dose is a
                    // convex combination of the 27 grid doses, so its distance from 0 is >= that of their range.
                    const float dr = fmaxf(fmaxf(dlo, -dhi), 0.0f);
                    const float outside2 = fminf(g.hmin2, fmaf(dr, dr, g.rho_link2));
                    if (key * key <= outside2) {          // nothing outside the star can be closer
                        out[lin] = key;
                        fused_stats_add(sStat, st, key);
                        toSearch = false;
                    } else {
                        key = fminf(key, sqrtf(vb));      // the 26 neighbour grid points also bound gamma from above
                    }
                }
            }
            if (!(key == key)) {                          // non-finite doses: no search, NaN out
                out[lin] = qnan;
                ++nNanKey;
                toSearch = false;
            }
        }
        // "ring" items: the star is done and what is left of the voxel's 2x2x2 block of cells decides (everything
        // else is at least hmin away); all other items walk the table from its first entry
        const bool deep = toSearch && classes && !(starDone && key * key < g.hmin2);
        const unsigned bal = __ballot_sync(FULL, toSearch && !deep);   // append to the work list, warp-aggregated
        if (bal) {
            const int leader = __ffs(bal) - 1;
            unsigned base = 0;
            if (lane == leader) base = atomicAdd(&ctl->nSearch, (unsigned)__popc(bal));
            base = __shfl_sync(FULL, base, leader);
            if (toSearch && !deep) {
                const unsigned pos = base + __popc(bal & ((1u << lane) - 1u));
                listKey[pos] = __float_as_uint(key);
                listIdx[pos] = (unsigned)lin;
                if (!classes) atomicAdd(&sHist[key_digit(key)], 1u);
                maxKey = fmaxf(maxKey, key);
            }
        }
        const unsigned balDeep = __ballot_sync(FULL, deep);
        if (balDeep) {
            const int leader = __ffs(balDeep) - 1;
            unsigned base = 0;
            if (lane == leader) base = atomicAdd(&ctl->nDeep, (unsigned)__popc(balDeep));
            base = __shfl_sync(FULL, base, leader);
            if (deep) {
                const unsigned pos = base + __popc(balDeep & ((1u << lane) - 1u));
                deepKey[pos] = __float_as_uint(key);
                deepIdx[pos] = (unsigned)lin;
                maxKey = fmaxf(maxKey, key);
            }
        }
        item = __shfl_sync(FULL, nextItem, 0);
        if (item < numItems && item * 32u + lane < M) linAhead = evalIdx[item * 32u + lane];
    }
    maxKey = warp_max(maxKey);
    if (lane == 0) sMax[tid >> 5] = maxKey;
    __syncthreads();
    if (!classes)
        for (int d = tid; d < KEY_DIGITS; d += STAR_THREADS)
            if (sHist[d]) atomicAdd(&ctl->hist[d], sHist[d]);
    if (tid == 0) {
        float m = 0.0f;
#pragma unroll
        for (int w = 0; w < STAR_THREADS / 32; ++w) m = fmaxf(m, sMax[w]);
        if (m > 0.0f) atomicMax(&ctl->maxKeyBits, __float_as_uint(m));
    }
    if (st.hist && nNanKey) atomicAdd(&st.summary->n_nan, nNanKey);
    fused_stats_flush(sStat, st);
    trace_last(e.call, 2);
}

// ------------------------------------------------------------------------------------------------
// a2: one-pass MSD radix presort of the search work list on the 8-bit key digit.  The digit histogram
// was accumulated by k_star; every block scans it (256 values) and scatters its share of the list.
// Order inside a digit is arbitrary (the search result does not depend on the order of the list).
// ------------------------------------------------------------------------------------------------
constexpr int SCATTER_THREADS = 256;

__global__ void __launch_bounds__(SCATTER_THREADS)
k_bucket_scatter(Ctl* __restrict__ ctl, const unsigned* __restrict__ keyIn, const unsigned* __restrict__ idxIn,
                 unsigned* __restrict__ keyOut, unsigned* __restrict__ idxOut)
{
    __shared__ unsigned sBase[KEY_DIGITS];
    __shared__ unsigned sWarp[SCATTER_THREADS / 32];
    const unsigned FULL = 0xffffffffu;
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    pdl_launch_dependents();
    pdl_wait();
    const unsigned n = ctl->nSearch;
    if (blockIdx.x * SCATTER_THREADS >= n) return;
    {   // exclusive scan of the 256-bin histogram
        const unsigned h = ctl->hist[tid];
        unsigned incl = h;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const unsigned t = __shfl_up_sync(FULL, incl, s);
            if (lane >= (unsigned)s) incl += t;
        }
        if (lane == 31) sWarp[warp] = incl;
        __syncthreads();
        unsigned off = 0;
        for (unsigned w = 0; w < warp; ++w) off += sWarp[w];
        sBase[tid] = off + incl - h;
        __syncthreads();
    }
    for (unsigned i0 = blockIdx.x * SCATTER_THREADS; i0 < n; i0 += gridDim.x * SCATTER_THREADS) {
        const unsigned i = i0 + tid;
        const bool valid = i < n;
        unsigned key = 0, idx = 0, d = KEY_DIGITS;            // invalid lanes form their own match group
        if (valid) { key = keyIn[i]; idx = idxIn[i]; d = key_digit(__uint_as_float(key)); }
        const unsigned peers = __match_any_sync(FULL, d);
        const int leader = __ffs(peers) - 1;
        unsigned base = 0;
        if (valid && (int)lane == leader) base = atomicAdd(&ctl->cursor[d], (unsigned)__popc(peers));
        base = __shfl_sync(FULL, base, leader);
        if (valid) {
            const unsigned pos = sBase[d] + base + __popc(peers & ((1u << lane) - 1u));
            keyOut[pos] = key;
            idxOut[pos] = idx;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a4: table search
// ------------------------------------------------------------------------------------------------
struct VoxelCtx {
    int v[3];
    int lin;
    float Dr, invdD;
    int algo;         // EvalP::algo
};

// Offset-dependent terms of the 26 faces owned by the vertex at (real-valued) offset (fx, fy, fz) voxels from the
// reference point (features_generated.cuh, gamma_owned_min): lam[T] = -(p . h_T) / A_T, q[a] = p_a^2, X[T].
// usable: bit a set when the owner's neighbour along +a is inside the grid.  A face that steps along an unusable axis
// does not exist (reading 11): lam[T] is NaN for every T holding such an axis, which fails the face's first comparison.
__device__ __forceinline__ void owned_face_terms(const GridP& g, float fx, float fy, float fz, unsigned usable,
                                                 float (&lam)[8], float (&q)[3], float (&X)[8])
{
    const float qnan = __int_as_float(0x7fc00000);
    const float px = fx * g.h[0], py = fy * g.h[1], pz = fz * g.h[2];
    q[0] = px * px; q[1] = py * py; q[2] = pz * pz;
    const float gx = (usable & 1u) ? fx : qnan, gy = (usable & 2u) ? fy : qnan, gz = (usable & 4u) ? fz : qnan;
    const float bxh = gx * g.hh[0], byh = gy * g.hh[1], bzh = gz * g.hh[2];
    lam[0] = 0.0f;
    lam[1] = -gx; lam[2] = -gy; lam[4] = -gz;
    lam[3] = -(bxh + byh) * g.invA[3];
    lam[5] = -(bxh + bzh) * g.invA[5];
    lam[6] = -(byh + bzh) * g.invA[6];
    lam[7] = -(bxh + byh + bzh) * g.invA[7];
    const float dxy = fx - fy, dxz = fx - fz, dyz = fy - fz;
    X[0] = X[1] = X[2] = X[4] = 0.0f;
    X[3] = g.K3 * dxy * dxy;
    X[5] = g.K5 * dxz * dxz;
    X[6] = g.K6 * dyz * dyz;
    X[7] = g.Kxy7 * dxy * dxy + g.Kyz7 * dyz * dyz + g.Kzx7 * dxz * dxz;
}

// All 26 faces owned by the grid vertex c = v + o; returns the new best^2.
template <bool JU>
__device__ __forceinline__ float eval_owner_vertex(const float* __restrict__ ev, const GridP& g, const VoxelCtx& vc,
                                                   int ox, int oy, int oz, float best2)
{
    const int cx = vc.v[0] + ox, cy = vc.v[1] + oy, cz = vc.v[2] + oz;
    if ((unsigned)cx >= (unsigned)g.n[0] || (unsigned)cy >= (unsigned)g.n[1] || (unsigned)cz >= (unsigned)g.n[2])
        return best2;                                          // vertex outside the grid (reading 11)
    const unsigned usable = (cx + 1 < g.n[0] ? 1u : 0u) | (cy + 1 < g.n[1] ? 2u : 0u) | (cz + 1 < g.n[2] ? 4u : 0u);
    const int sx = (usable & 1u) ? 1 : 0, sy = (usable & 2u) ? g.stride[1] : 0, sz = (usable & 4u) ? g.stride[2] : 0;
    const float* p = ev + (vc.lin + ox + oy * g.stride[1] + oz * g.stride[2]);
    if (vc.algo == 1) {                                        // classical discrete search (Low et al.): vertex c only
        const float dv = (__ldg(p) - vc.Dr) * vc.invdD;
        const float fx0 = (float)ox * g.h[0], fy0 = (float)oy * g.h[1], fz0 = (float)oz * g.h[2];
        return fminf(best2, fmaf(dv, dv, fmaf(fx0, fx0, fmaf(fy0, fy0, fz0 * fz0))));
    }
    float d[8];
#pragma unroll
    for (int S = 0; S < 8; ++S)                                // 32-bit offsets from one base pointer
        d[S] = (__ldg(p + (((S & 1) ? sx : 0) + ((S & 2) ? sy : 0) + ((S & 4) ? sz : 0))) - vc.Dr) * vc.invdD;
    if (JU && vc.algo == 2) {                                  // variant: whole cells by the recursion of PAPER.md:209
        if (usable != 7u) return best2;                        // only cells fully inside the grid exist (reading 11)
        return ju_cell_min(d, g, ox, oy, oz, best2);
    }
    float lam[8], q[3], X[8];
    owned_face_terms(g, (float)ox, (float)oy, (float)oz, usable, lam, q, X);
    return gamma_owned_min(d, g.invA, lam, q, X, best2);
}

template <int G>
__device__ __forceinline__ float group_min(float v)
{
#pragma unroll
    for (int s = G / 2; s > 0; s >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}

#ifndef GAMMA_SEARCH_THREADS
#define GAMMA_SEARCH_THREADS 128
#endif
#ifndef GAMMA_SEARCH_MIN_BLOCKS
#define GAMMA_SEARCH_MIN_BLOCKS 6
#endif
constexpr int SEARCH_THREADS = GAMMA_SEARCH_THREADS;
constexpr int SEARCH_MIN_BLOCKS = GAMMA_SEARCH_MIN_BLOCKS;   // adaptive-lane kernel (MODE 0): register budget
#ifndef GAMMA_SEARCH_GRID_BLOCKS
#define GAMMA_SEARCH_GRID_BLOCKS GAMMA_SEARCH_MIN_BLOCKS
#endif
constexpr int SEARCH_GRID_BLOCKS = GAMMA_SEARCH_GRID_BLOCKS; // blocks per SM actually launched (<= SEARCH_MIN_BLOCKS)

struct SearchCtx {
    const float* ref; const float* ev; float* out;
    const int4* table;
    unsigned T;
    bool trunc;
    float Rtab2, invGlobal;
    double dnorm;
    FusedStats<SEARCH_THREADS>* stat;   // a6 fused (gamma_opts::stats_*)
    StatsP st;
};

// One warp searches 32/G consecutive work items (firstItem .. firstItem + 32/G - 1, counted from the END of the
// sorted list: deepest first), G lanes per reference voxel.  Returns the owner vertices it evaluated.
template <int G, bool JU = false>
__device__ __forceinline__ unsigned search_items(const SearchCtx& c, const GridP& g, const EvalP& e,
                                                 const unsigned* __restrict__ listKey,
                                                 const unsigned* __restrict__ listIdx, unsigned nList,
                                                 unsigned firstItem, int lane, bool pre = false, unsigned preIdx = 0u,
                                                 unsigned preKey = 0u)
{
    // pre: (preIdx, preKey) is this lane's list entry, fetched while the previous work item was searched
    constexpr int EPP = G >= 8 ? G / 8 : 1;     // table entries per pass
    const unsigned FULL = 0xffffffffu;
    const int gid = lane / G, gl = lane % G;
    const unsigned item = firstItem + gid;
    const bool have = item < nList;
    const unsigned T = c.T;
    unsigned visits = 0;
    VoxelCtx vc;
    float key = 0.0f, best2 = 0.0f;
    if (have) {
        const unsigned idx = nList - 1u - item;
        vc.lin = (int)(pre ? preIdx : listIdx[idx]);
        key = __uint_as_float(pre ? preKey : listKey[idx]);
        vc.Dr = __ldg(c.ref + vc.lin);
        vc.invdD = e.mode == 0 ? c.invGlobal : criterion_inv_dD(e, c.dnorm, vc.Dr);
        voxel_coords(g, vc.lin, vc.v[0], vc.v[1], vc.v[2]);
        vc.algo = e.algo;
        best2 = key * key;
    } else {
        vc.lin = 0; vc.Dr = 0.0f; vc.invdD = 0.0f; vc.v[0] = vc.v[1] = vc.v[2] = 0; vc.algo = e.algo;
    }
    // ---- Algorithm A1 step 4-b over the sorted table
    for (unsigned e0 = 0;; e0 += EPP) {
        bool more = have && e0 < T;
        if (more) more = __int_as_float(__ldg(&c.table[e0].x)) < best2;    // 4-b-ii: stop at L >= gamma
        if (!__any_sync(FULL, more)) break;
        if (G >= 8) {
            const unsigned en = e0 + (unsigned)(gl >> 3);
            float cand = best2;
            if (more && en < T) {
                const int4 t = __ldg(&c.table[en]);
                if (__int_as_float(t.x) < best2) {
                    const int ox = (gl & 1) ? -t.y - 1 : t.y;
                    const int oy = (gl & 2) ? -t.z - 1 : t.z;
                    const int oz = (gl & 4) ? -t.w - 1 : t.w;
                    cand = eval_owner_vertex<JU>(c.ev, g, vc, ox, oy, oz, best2);
                    ++visits;
                }
            }
            best2 = group_min<(G >= 8 ? G : 8)>(cand);
        } else {
            if (more) {
                const int4 t = __ldg(&c.table[e0]);
#pragma unroll 1
                for (int var = 0; var < 8; ++var) {
                    const int ox = (var & 1) ? -t.y - 1 : t.y;
                    const int oy = (var & 2) ? -t.z - 1 : t.z;
                    const int oz = (var & 4) ? -t.w - 1 : t.w;
                    best2 = eval_owner_vertex<JU>(c.ev, g, vc, ox, oy, oz, best2);
                    ++visits;
                }
            }
        }
    }
    // ---- beyond a truncated (prefix) table: Chebyshev shells of octant cells, sh = max(m_x, m_y, m_z) = 0, 1, 2, ...
    // Every cell of shell sh has some m_a = sh, so nothing in it is closer than sh * hmin: the walk stops at the first
    // shell with (sh * hmin)^2 >= gamma^2 -- it reaches as far as the running gamma, not as far as the key, and
    // there is no radius cap.  Cells the table already covered (L^2 < Rtab^2) are skipped.
    if (c.trunc) {
        const float Rtab2 = c.Rtab2;
        const int shMax = max(g.n[0], max(g.n[1], g.n[2])) - 1;
        for (int sh = 0; sh <= shMax; ++sh) {
            const bool go = have && best2 > Rtab2 && (float)sh * (float)sh * g.hmin2 < best2;
            if (!__any_sync(FULL, go)) break;
            // the shell as three slabs: m_x = sh | m_y = sh, m_x < sh | m_z = sh, m_x < sh, m_y < sh (clipped to the grid)
            const int ey = min(sh, g.n[1] - 1), ez = min(sh, g.n[2] - 1);
            const int exm = min(sh - 1, g.n[0] - 1), eym = min(sh - 1, g.n[1] - 1);
            const unsigned cX = sh <= g.n[0] - 1 ? (unsigned)((ey + 1) * (ez + 1)) : 0u;
            const unsigned cY = (sh >= 1 && sh <= g.n[1] - 1) ? (unsigned)((exm + 1) * (ez + 1)) : 0u;
            const unsigned cZ = (sh >= 1 && sh <= g.n[2] - 1) ? (unsigned)((exm + 1) * (eym + 1)) : 0u;
            const unsigned V = cX + cY + cZ;
            auto cell_of = [&](unsigned i, int& mx, int& my, int& mz) {
                if (i < cX) { mx = sh; my = (int)(i % (unsigned)(ey + 1)); mz = (int)(i / (unsigned)(ey + 1)); }
                else if (i < cX + cY) { const unsigned j = i - cX; my = sh; mx = (int)(j % (unsigned)(exm + 1)); mz = (int)(j / (unsigned)(exm + 1)); }
                else { const unsigned j = i - cX - cY; mz = sh; mx = (int)(j % (unsigned)(exm + 1)); my = (int)(j / (unsigned)(exm + 1)); }
            };
            for (unsigned i0 = 0; i0 < V; i0 += EPP) {
                if (G >= 8) {
                    const unsigned i = i0 + (unsigned)(gl >> 3);
                    float cand = best2;
                    if (go && i < V) {
                        int mx, my, mz;
                        cell_of(i, mx, my, mz);
                        const float L2 = cell_L2(mx, my, mz, g);
                        if (L2 >= Rtab2 && L2 < best2) {
                            const int ox = (gl & 1) ? -mx - 1 : mx;
                            const int oy = (gl & 2) ? -my - 1 : my;
                            const int oz = (gl & 4) ? -mz - 1 : mz;
                            cand = eval_owner_vertex<JU>(c.ev, g, vc, ox, oy, oz, best2);
                            ++visits;
                        }
                    }
                    best2 = group_min<(G >= 8 ? G : 8)>(cand);
                } else if (go) {
                    int mx, my, mz;
                    cell_of(i0, mx, my, mz);
                    const float L2 = cell_L2(mx, my, mz, g);
                    if (L2 >= Rtab2 && L2 < best2) {
#pragma unroll 1
                        for (int var = 0; var < 8; ++var) {
                            const int ox = (var & 1) ? -mx - 1 : mx;
                            const int oy = (var & 2) ? -my - 1 : my;
                            const int oz = (var & 4) ? -mz - 1 : mz;
                            best2 = eval_owner_vertex<JU>(c.ev, g, vc, ox, oy, oz, best2);
                            ++visits;
                        }
                    }
                }
            }
        }
    }
    if (have && gl == 0) {
        const float gam = fminf(key, sqrtf(best2));
        c.out[vc.lin] = gam;                                         // a5: write at the voxel's own place
        fused_stats_add(*c.stat, c.st, gam);
    }
    return visits;
}

// One thread per "ring" item (depth classes): an interior voxel whose star phase is done and whose running
// gamma is below the smallest voxel spacing.  Everything that can still be closer lies in the 72 ring faces of its
// 2x2x2 block of cells (gamma_ring_min); the 27 doses are re-read (L1/L2 hits) and no table is walked.
__device__ __forceinline__ void ring_items(const SearchCtx& c, const GridP& g, const EvalP& e, const GammaRingP& R,
                                           const unsigned* __restrict__ listKey,
                                           const unsigned* __restrict__ listIdx, unsigned nList, unsigned firstItem,
                                           int lane, bool pre = false, unsigned preIdx = 0u, unsigned preKey = 0u)
{
    const unsigned item = firstItem + (unsigned)lane;
    if (item >= nList) return;
    const int lin = (int)(pre ? preIdx : listIdx[item]);
    const float key = __uint_as_float(pre ? preKey : listKey[item]);
    const float Dr = __ldg(c.ref + lin);
    const float invdD = e.mode == 0 ? c.invGlobal : criterion_inv_dD(e, c.dnorm, Dr);
    const float* p = c.ev + lin;
    float d[27];
#pragma unroll
    for (int oz = -1; oz <= 1; ++oz)
#pragma unroll
        for (int oy = -1; oy <= 1; ++oy)
#pragma unroll
            for (int ox = -1; ox <= 1; ++ox)
                d[(ox + 1) + 3 * (oy + 1) + 9 * (oz + 1)] =
                    (__ldg(p + ox + oy * g.stride[1] + oz * g.stride[2]) - Dr) * invdD;
    const float best2 = gamma_ring_min(d, g.invA, R, key * key);
    const float gam = fminf(key, sqrtf(best2));
    c.out[lin] = gam;                                      // a5: write at the voxel's own place
    fused_stats_add(*c.stat, c.st, gam);
}

// MODE = lanes per reference voxel: 1 (thread per voxel), 8, 32, or 0 = adaptive: deep items (the
// walk will pass the first table entry) get a whole warp each, the others 8 lanes each.  Deep items are either
// the tail of the sorted list (key digit >= deepDigit, counted from the digit histogram) or, with depth-class
// lists (classes != 0), the separate list (deepKey, deepIdx) that k_star filled; the other list then holds "ring"
// items only, searched one per thread (ring_items).  Work units are handed out
// deepest first: first round static, later rounds by an atomic counter whose latency hides behind the search.
// JU: the instantiation that also holds the recursion variant (ju_simplex.cuh); kept out of the default kernels, whose
// register allocation it would disturb.
template <int MODE, bool JU = false>
__global__ void __launch_bounds__(SEARCH_THREADS, (MODE == 0 && !JU) ? SEARCH_MIN_BLOCKS : 1)
k_table_search(const float* __restrict__ ref, const float* __restrict__ ev, float* __restrict__ out, GridP g,
               EvalP e, Ctl* __restrict__ ctl, const unsigned* __restrict__ listKey,
               const unsigned* __restrict__ listIdx, const unsigned* __restrict__ deepKey,
               const unsigned* __restrict__ deepIdx, const int4* __restrict__ table, int deepDigit, int classes,
               const __grid_constant__ GammaRingP ring, StatsP st)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    __shared__ FusedStats<SEARCH_THREADS> sStat;
    SearchCtx c;
#ifdef GAMMA_TRACE
    TraceWarp tw;
    tw.start = trace_now(); tw.waited = 0; tw.firstUnit = 0; tw.end = 0; tw.units = 0;
#endif
    fused_stats_init(sStat, st);
    trace_first(e.call, 3);
    pdl_wait();
    pdl_launch_dependents();                             // the next call's k_norm may use the SMs this kernel leaves
    trace_waited(e.call, 3);
#ifdef GAMMA_TRACE
    tw.waited = trace_now();
#endif
    const unsigned nS = ctl->nSearch;
    unsigned nDeep = 0;
    if (MODE == 0 && classes) {
        nDeep = ctl->nDeep;
    } else if (MODE == 0 && deepDigit < KEY_DIGITS) {         // sum of the histogram tail = number of deep items
        for (int d = deepDigit + lane; d < KEY_DIGITS; d += 32) nDeep += ctl->hist[d];
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) nDeep += __shfl_xor_sync(FULL, nDeep, s);
        deepKey = listKey; deepIdx = listIdx;
    }
    // shallow items: all of the list with depth classes, else what is left of the sorted list before its deep tail
    const unsigned nShallow = (MODE == 0 && classes) ? nS : nS - nDeep;
    const unsigned nDeepList = (MODE == 0 && classes) ? nDeep : nS;   // deep item i is entry nDeepList - 1 - i
    constexpr unsigned VPW = MODE == 0 ? 4u : 32u / (unsigned)(MODE == 0 ? 8 : MODE);
    const unsigned numUnits = MODE != 0 ? (nS + VPW - 1u) / VPW
                              : classes ? nDeep + (nShallow + 31u) / 32u : nDeep + (nShallow + 3u) / 4u;
    const unsigned warpsTotal = gridDim.x * (SEARCH_THREADS / 32);
    unsigned unit = blockIdx.x * (SEARCH_THREADS / 32) + (threadIdx.x >> 5);
    if (unit < numUnits) {
        // whole rounds are static (k_star); a last partial round of less than half of the warps goes by tickets, a larger
        // one is static too (thousands of tickets from one address cost more than the imbalance they would repair)
        unsigned staticRounds = numUnits / warpsTotal;
        const bool tickets = staticRounds && 2u * (numUnits - staticRounds * warpsTotal) < warpsTotal;
        if (!tickets) ++staticRounds;
        const unsigned one = ticket_one(ctl);
        unsigned round = 1;
        c.ref = ref; c.ev = ev; c.out = out; c.table = table;
        c.T = ctl->tableCount;
        c.trunc = ctl->tableTrunc != 0;
        c.Rtab2 = ctl->Rtab2;
        const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
        c.dnorm = (double)dnormF;
        c.invGlobal = ctl->invGlobal;
        c.stat = &sStat; c.st = st;
        unsigned visits = 0;
        bool pre = false;
        unsigned preIdx = 0u, preKey = 0u;

        while (unit < numUnits) {
            unsigned nextUnit = numUnits;
            const bool staticNext = round < staticRounds;
            if (staticNext) nextUnit = unit + warpsTotal;
            else if (tickets && lane == 0) nextUnit = ticket_next(&ctl->workCounter, one) + staticRounds * warpsTotal;
            ++round;
            // the list entry of a statically known next unit is fetched now and used after this unit's search
            const bool havePre = pre;
            const unsigned curIdx = preIdx, curKey = preKey;
            pre = false;
            if (MODE == 0 && classes && staticNext) {
                if (nextUnit < nDeep) {
                    const unsigned idx = nDeepList - 1u - nextUnit;
                    preIdx = deepIdx[idx]; preKey = deepKey[idx]; pre = true;
                } else {
                    const unsigned item = 32u * (nextUnit - nDeep) + (unsigned)lane;
                    if (item < nS) { preIdx = listIdx[item]; preKey = listKey[item]; }
                    pre = true;
                }
            }
            if (MODE == 0) {
                if (unit < nDeep) visits += search_items<32, JU>(c, g, e, deepKey, deepIdx, nDeepList, unit, lane, havePre, curIdx, curKey);
                else if (classes) ring_items(c, g, e, ring, listKey, listIdx, nS, 32u * (unit - nDeep), lane, havePre, curIdx, curKey);
                else visits += search_items<8, JU>(c, g, e, listKey, listIdx, nS, nDeep + 4u * (unit - nDeep), lane);
            } else {
                visits += search_items<(MODE == 0 ? 8 : MODE), JU>(c, g, e, listKey, listIdx, nS, unit * VPW, lane);
            }
            unit = __shfl_sync(FULL, nextUnit, 0);
#ifdef GAMMA_TRACE
            if (tw.units++ == 0) tw.firstUnit = trace_now();
#endif
        }
        // diagnostic counter: one atomic per warp
        for (int s = 16; s > 0; s >>= 1) visits += __shfl_xor_sync(FULL, visits, s);
        if (lane == 0 && visits) atomicAdd(&ctl->visits, (unsigned long long)visits);
    }
    fused_stats_flush(sStat, st);
#ifdef GAMMA_TRACE
    {
        const unsigned wid = blockIdx.x * (SEARCH_THREADS / 32) + (threadIdx.x >> 5);
        tw.end = trace_now();
        if (lane == 0 && g_trace_warps && wid < TRACE_WARPS) g_trace_warps[wid] = tw;
    }
#endif
    trace_last(e.call, 3);
}

}  // namespace gamma_b200
