// offset_table.cuh -- subsystem (1): the radially pre-sorted offset table {n, L_n}
// (Algorithm A1 steps 2-3; Algorithm A2 steps 4-5; Wendling's
// pre-sort), with two changes explained in DESIGN.md:
//   * the bound of an offset is the minimum spatial distance of its CELL, L(o)^2 = sum_a (m_a h_a)^2 with
//     m_a = max(o_a, -o_a-1) (reading 4), not the distance of the voxel (i,j,k) of PAPER.md:180;
//   * L(o) depends on m only, so the table lists the octant m >= 0 and the search expands an entry into
//     its 8 offsets o_a in {m_a, -m_a-1}: 8x fewer entries to generate and sort.
// The radius is max key of the search list, known only on the device; the kernel reads it there.
//
// One block: (1) bucket histogram of L^2 over the candidate box, (2) scan, (3) scatter into buckets,
// (4) exact rank inside each bucket by (L^2 bits, box index) -> a fully and deterministically sorted
// table.  A counting sort fits because the table is small (10^1..10^5 entries).
#pragma once
#include "common.cuh"

namespace gamma_b200 {

constexpr int TAB_THREADS = 1024;
constexpr int TAB_BUCKETS = 4096;

// radius_in >= 0: use it; < 0: radius = largest key of the search list (ctl->maxKeyBits).
__global__ void __launch_bounds__(TAB_THREADS)
k_offset_table(GridP g, Ctl* __restrict__ ctl, float radius_in, long long cap, int4* __restrict__ table,
               unsigned* __restrict__ tmpL, unsigned* __restrict__ tmpIdx)
{
    __shared__ unsigned start[TAB_BUCKETS + 1];
    __shared__ unsigned cursor[TAB_BUCKETS];
    __shared__ unsigned warpSums[32];
    __shared__ float sR2, sScale;
    __shared__ int sBox[3];
    __shared__ unsigned sTrunc;
    const unsigned tid = threadIdx.x;

    if (tid == 0) {
        float R = radius_in >= 0.0f ? radius_in : __uint_as_float(ctl->maxKeyBits);
        if (!(R >= 0.0f)) R = 0.0f;                    // NaN guard
        unsigned trunc = 0;
        int bx, by, bz;
        for (;;) {
            bx = g.h[0] > 0.0f ? (int)fminf((float)(g.n[0] - 1), floorf(R / g.h[0])) + 1 : 1;
            by = g.h[1] > 0.0f ? (int)fminf((float)(g.n[1] - 1), floorf(R / g.h[1])) + 1 : 1;
            bz = g.h[2] > 0.0f ? (int)fminf((float)(g.n[2] - 1), floorf(R / g.h[2])) + 1 : 1;
            if ((long long)bx * by * bz <= cap) break;
            // an in-grid box that is already as large as the grid cannot shrink by lowering R slowly;
            // 0.8 per step terminates because cap >= 1 and R -> 0 gives a 1x1x1 box.
            R *= 0.8f;
            trunc = 1;
        }
        sBox[0] = bx; sBox[1] = by; sBox[2] = bz;
        sR2 = R * R;
        sScale = R > 0.0f ? (float)TAB_BUCKETS / (R * R) : 0.0f;
        sTrunc = trunc;
    }
    for (unsigned b = tid; b < TAB_BUCKETS; b += TAB_THREADS) cursor[b] = 0;
    __syncthreads();
    const int bx = sBox[0], by = sBox[1], bz = sBox[2];
    const unsigned V = (unsigned)(bx * by * bz);
    const float R2 = sR2, scale = sScale;

    // (1) histogram
    for (unsigned i = tid; i < V; i += TAB_THREADS) {
        const int mx = i % bx, my = (i / bx) % by, mz = i / (bx * by);
        const float L2 = cell_L2(mx, my, mz, g);
        if (L2 < R2) atomicAdd(&cursor[min(TAB_BUCKETS - 1, (int)(L2 * scale))], 1u);
    }
    __syncthreads();
    // (2) exclusive scan of the 4096 bucket counts (4 per thread)
    {
        unsigned c[4], s = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) { c[j] = cursor[tid * 4 + j]; s += c[j]; }
        const unsigned lane = tid & 31u, warp = tid >> 5;
        unsigned incl = s;
#pragma unroll
        for (int k = 1; k < 32; k <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, incl, k);
            if (lane >= (unsigned)k) incl += t;
        }
        if (lane == 31) warpSums[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            unsigned w = warpSums[lane], wi = w;
#pragma unroll
            for (int k = 1; k < 32; k <<= 1) {
                const unsigned t = __shfl_up_sync(0xffffffffu, wi, k);
                if (lane >= (unsigned)k) wi += t;
            }
            warpSums[lane] = wi - w;
        }
        __syncthreads();
        unsigned run = warpSums[warp] + incl - s;
#pragma unroll
        for (int j = 0; j < 4; ++j) { start[tid * 4 + j] = run; cursor[tid * 4 + j] = run; run += c[j]; }
        if (tid == TAB_THREADS - 1) start[TAB_BUCKETS] = run;
    }
    __syncthreads();
    const unsigned T = start[TAB_BUCKETS];
    // (3) scatter into buckets (order inside a bucket is arbitrary here)
    for (unsigned i = tid; i < V; i += TAB_THREADS) {
        const int mx = i % bx, my = (i / bx) % by, mz = i / (bx * by);
        const float L2 = cell_L2(mx, my, mz, g);
        if (L2 < R2) {
            const unsigned pos = atomicAdd(&cursor[min(TAB_BUCKETS - 1, (int)(L2 * scale))], 1u);
            tmpL[pos] = __float_as_uint(L2);
            tmpIdx[pos] = i;
        }
    }
    __syncthreads();   // block-wide visibility of the global writes above (single block)
    // (4) exact rank inside the bucket
    for (unsigned i = tid; i < T; i += TAB_THREADS) {
        const unsigned Lb = tmpL[i], id = tmpIdx[i];
        const int b = min(TAB_BUCKETS - 1, (int)(__uint_as_float(Lb) * scale));
        const unsigned lo = start[b], hi = start[b + 1];
        unsigned rank = 0;
        for (unsigned j = lo; j < hi; ++j) {
            const unsigned Lj = tmpL[j];
            rank += (Lj < Lb) || (Lj == Lb && tmpIdx[j] < id);
        }
        const int mx = id % bx, my = (id / bx) % by, mz = id / (bx * by);
        table[lo + rank] = make_int4((int)Lb, mx, my, mz);
    }
    if (tid == 0) {
        ctl->tableCount = T;
        ctl->tableTrunc = sTrunc;
        ctl->Rtab2 = R2;
        ctl->box[0] = bx; ctl->box[1] = by; ctl->box[2] = bz;
    }
}

}  // namespace gamma_b200
