// offset_table.cuh -- subsystem (1): the radially pre-sorted offset table {n, L_n}
// (Algorithm A1 steps 2-3; Algorithm A2 steps 4-5; Wendling's
// pre-sort), with two changes explained in DESIGN.md:
//   * the bound of an offset is the minimum spatial distance of its CELL, L(o)^2 = sum_a (m_a h_a)^2 with
//     m_a = max(o_a, -o_a-1) (reading 4), not the distance of the voxel (i,j,k) of PAPER.md:180;
//   * L(o) depends on m only, so the table lists the octant m >= 0 and the search expands an entry into
//     its 8 offsets o_a in {m_a, -m_a-1}: 8x fewer entries to generate and sort.
// The radius is the paper's: max |DD| / dD (A1 step 1), read from the control block that
// k_norm filled, so the table is built concurrently with the prep/star kernel.
//
// Counting sort on 4096 linear buckets of L^2, finished by an exact rank inside each bucket by
// (L^2 bits, box index): a fully and deterministically sorted table.  TAB_BLOCKS blocks work without talking
// to each other: every block histograms the whole candidate box (cheap integer work) and then collects,
// ranks and writes only its own slice of 4096 / TAB_BLOCKS buckets, from shared memory when the slice fits.
#pragma once
#include "common.cuh"

namespace gamma_b200 {

constexpr int TAB_THREADS = 1024;
constexpr int TAB_BUCKETS = 4096;
constexpr int TAB_BLOCKS = 32;
constexpr int TAB_SLICE = TAB_BUCKETS / TAB_BLOCKS;      // buckets finished by one block
constexpr int TAB_SMEM_ENTRIES = 8192;                   // slice entries kept in shared memory (else global scratch)
constexpr size_t TAB_DYN_SMEM = (size_t)TAB_SMEM_ENTRIES * 2 * sizeof(unsigned);

// Diagonal of the grid in DTA units: nothing is farther away than this.
__host__ __device__ inline float grid_diagonal(const GridP& g)
{
    const float ax = (float)(g.n[0] - 1) * g.h[0], ay = (float)(g.n[1] - 1) * g.h[1], az = (float)(g.n[2] - 1) * g.h[2];
    return sqrtf(ax * ax + ay * ay + az * az) * 1.0001f + 1e-3f;
}

// Cells of the candidate box of radius R (m_a in [0, box_a)), the quantity `cap` limits.
__host__ __device__ inline long long table_box_cells(const GridP& g, float R, int& bx, int& by, int& bz)
{
    bx = g.h[0] > 0.0f ? (int)fminf((float)(g.n[0] - 1), floorf(R / g.h[0])) + 1 : 1;
    by = g.h[1] > 0.0f ? (int)fminf((float)(g.n[1] - 1), floorf(R / g.h[1])) + 1 : 1;
    bz = g.h[2] > 0.0f ? (int)fminf((float)(g.n[2] - 1), floorf(R / g.h[2])) + 1 : 1;
    return (long long)bx * by * bz;
}

// Upper bound of every key of the search list (the paper's table radius max(DD)/dD), from k_norm's maxima.
__device__ inline float table_radius_from_ctl(const GridP& g, const EvalP& e, const Ctl* ctl)
{
    const float dnormF = e.norm_dose > 0.0f ? e.norm_dose : ordered_to_float(ctl->normOrd);
    const double dnorm = (double)dnormF;
    const float maxAbs = __uint_as_float(ctl->maxAbsDD);
    float R;
    if (e.mode == 0) {
        const double dD = (double)e.DD * dnorm;
        R = dD > 0.0 ? maxAbs * (float)(1.0 / dD) : 0.0f;            // same rounding as the keys: monotone bound
    } else {
        double r = (double)__uint_as_float(ctl->maxRatio) / (double)e.DD;
        const double floorD = (double)e.cutoff * dnorm;               // evaluated voxels have D_r >= cutoff * D_norm
        if (floorD > 0.0) r = fmin(r, (double)maxAbs / ((double)e.DD * floorD));
        R = (float)(r * (1.0 + 1e-5)) + 1e-30f;
    }
    if (!(R >= 0.0f)) R = 0.0f;                                       // NaN guard
    // nothing in the grid is farther than its diagonal: clamp (also makes an infinite bound finite)
    return fminf(R, grid_diagonal(g));
}

// radius_in >= 0: use it; < 0: radius from the control block (table_radius_from_ctl).
// prefix != 0: radius_in is a data-independent radius (as far as `cap` allows): the table is a PREFIX of the
// paper's table, flagged truncated unless it reaches the grid diagonal, and the search goes on beyond it by
// enumeration -- so the kernel needs nothing from k_norm and runs beside it.
__global__ void __launch_bounds__(TAB_THREADS)
k_offset_table(GridP g, EvalP e, Ctl* __restrict__ ctl, float radius_in, long long cap, int4* __restrict__ table,
               unsigned* __restrict__ tmpL, unsigned* __restrict__ tmpIdx, int prefix)
{
    extern __shared__ unsigned sSlice[];                 // [TAB_SMEM_ENTRIES] L^2 bits, [TAB_SMEM_ENTRIES] box index
    __shared__ unsigned start[TAB_BUCKETS + 1];
    __shared__ unsigned cursor[TAB_SLICE];
    __shared__ unsigned warpSums[32];
    __shared__ float sR2, sScale;
    __shared__ int sBox[3];
    __shared__ unsigned sTrunc;
    const unsigned tid = threadIdx.x;

    if (tid == 0) {
        float R = radius_in >= 0.0f ? radius_in : table_radius_from_ctl(g, e, ctl);
        if (!(R >= 0.0f)) R = 0.0f;
        R = fminf(R, 3.0e18f);
        unsigned trunc = (prefix && R < grid_diagonal(g)) ? 1u : 0u;
        int bx, by, bz;
        for (;;) {
            if (table_box_cells(g, R, bx, by, bz) <= cap) break;
            // 0.8 per step terminates because cap >= 1 and R -> 0 gives a 1x1x1 box
            R *= 0.8f;
            trunc = 1;
        }
        sBox[0] = bx; sBox[1] = by; sBox[2] = bz;
        sR2 = R * R;
        sScale = R > 0.0f ? (float)TAB_BUCKETS / (R * R) : 0.0f;
        sTrunc = trunc;
    }
    for (unsigned b = tid; b < TAB_BUCKETS; b += TAB_THREADS) start[b] = 0;
    __syncthreads();
    const int bx = sBox[0], by = sBox[1], bz = sBox[2];
    const unsigned V = (unsigned)(bx * by * bz);
    const float R2 = sR2, scale = sScale;
    auto bucket_of = [&](float L2) { return min(TAB_BUCKETS - 1, (int)(L2 * scale)); };

    // (1) histogram of the whole box (every block)
    for (unsigned i = tid; i < V; i += TAB_THREADS) {
        const int mx = i % bx, my = (i / bx) % by, mz = i / (bx * by);
        const float L2 = cell_L2(mx, my, mz, g);
        if (L2 < R2) atomicAdd(&start[bucket_of(L2)], 1u);
    }
    __syncthreads();
    // (2) exclusive scan of the 4096 bucket counts (4 per thread)
    {
        unsigned c[4], s = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) { c[j] = start[tid * 4 + j]; s += c[j]; }
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
        for (int j = 0; j < 4; ++j) { start[tid * 4 + j] = run; run += c[j]; }
        if (tid == TAB_THREADS - 1) start[TAB_BUCKETS] = run;
    }
    __syncthreads();
    const unsigned T = start[TAB_BUCKETS];
    // (3) this block's slice of buckets: collect its entries (order inside a bucket is arbitrary here)
    const int b0 = blockIdx.x * TAB_SLICE;
    const unsigned lo0 = start[b0], cnt = start[b0 + TAB_SLICE] - lo0;
    const bool inSmem = cnt <= (unsigned)TAB_SMEM_ENTRIES;
    unsigned* const Ls = inSmem ? sSlice : tmpL + lo0;
    unsigned* const Is = inSmem ? sSlice + TAB_SMEM_ENTRIES : tmpIdx + lo0;
    if (tid < TAB_SLICE) cursor[tid] = start[b0 + tid] - lo0;
    __syncthreads();
    if (cnt > 0) {
        for (unsigned i = tid; i < V; i += TAB_THREADS) {
            const int mx = i % bx, my = (i / bx) % by, mz = i / (bx * by);
            const float L2 = cell_L2(mx, my, mz, g);
            if (L2 < R2) {
                const int b = bucket_of(L2) - b0;
                if (b >= 0 && b < TAB_SLICE) {
                    const unsigned pos = atomicAdd(&cursor[b], 1u);
                    Ls[pos] = __float_as_uint(L2);
                    Is[pos] = i;
                }
            }
        }
    }
    __threadfence_block();
    __syncthreads();
    // (4) exact rank inside the bucket, write the final entry
    for (unsigned i = tid; i < cnt; i += TAB_THREADS) {
        const unsigned Lb = Ls[i], id = Is[i];
        const int b = bucket_of(__uint_as_float(Lb));
        const unsigned lo = start[b] - lo0, hi = start[b + 1] - lo0;
        unsigned rank = 0;
        for (unsigned j = lo; j < hi; ++j) {
            const unsigned Lj = Ls[j];
            rank += (Lj < Lb) || (Lj == Lb && Is[j] < id);
        }
        const int mx = id % bx, my = (id / bx) % by, mz = id / (bx * by);
        table[lo0 + lo + rank] = make_int4((int)Lb, mx, my, mz);
    }
    if (blockIdx.x == 0 && tid == 0) {
        ctl->tableCount = T;
        ctl->tableTrunc = sTrunc;
        ctl->Rtab2 = R2;
        ctl->box[0] = bx; ctl->box[1] = by; ctl->box[2] = bz;
    }
}

}  // namespace gamma_b200
