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
constexpr int TAB_BLOCKS = 32;                           // slices: blocks that each finish 4096 / 32 buckets
constexpr int TAB_SLICE = TAB_BUCKETS / TAB_BLOCKS;      // buckets finished by one block
constexpr int TAB_SMEM_ENTRIES = 8192;                   // slice entries kept in shared memory (else global scratch)
// the builder embedded in k_star (small prefix tables): 4 slices of a 1024-bucket counting sort, all entries in smem
constexpr long long TAB_EMBED_MAX_CELLS = 1024;          // largest candidate box the embedded builder takes
constexpr int TAB_EMBED_BUCKETS = 1024;
constexpr int TAB_EMBED_BLOCKS = 4;
constexpr int TAB_EMBED_ENTRIES = 1024;

// What a table build needs to know before it touches a cell: radius, candidate box, bucket scale, and the magic
// numbers of the exact division by box_x (0) and box_x * box_y (1) (fast_div).  Made on the host when the radius is
// data-independent, else by thread 0 of every building block.
struct TablePlan {
    float R2, scale;
    int box[3];
    unsigned trunc;
    unsigned divMul[2], divSh[2];
};

// Shared-memory working set of one table-building block: NB buckets, NS slices, ENT slice entries in smem.
template <int ENT, int NB, int NS>
struct TableSmem {
    unsigned start[NB + 1];
    unsigned cursor[NB / NS];
    unsigned warpSums[32];
    unsigned slice[2 * ENT];                             // [ENT] L^2 bits, [ENT] box index
    TablePlan plan;
};
constexpr size_t TAB_DYN_SMEM = sizeof(TableSmem<TAB_SMEM_ENTRIES, TAB_BUCKETS, TAB_BLOCKS>);

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

// prefix != 0: R is a data-independent radius: the table is flagged truncated unless it reaches the grid diagonal.
__host__ __device__ inline TablePlan table_plan_make(const GridP& g, float R, long long cap, int prefix, int buckets)
{
    TablePlan P;
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
    P.box[0] = bx; P.box[1] = by; P.box[2] = bz;
    const unsigned dv[2] = {(unsigned)bx, (unsigned)(bx * by)};
    for (int k = 0; k < 2; ++k) {                        // same magic numbers as GridP::divMul (box cells < 2^31)
        unsigned l = 0;
        while ((1ull << l) < dv[k]) ++l;
        P.divMul[k] = (unsigned)((1ull << (31 + l)) / dv[k] + 1ull);
        P.divSh[k] = 31 + l;
    }
    P.R2 = R * R;
    P.scale = R > 0.0f ? (float)buckets / (R * R) : 0.0f;
    P.trunc = trunc;
    return P;
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

// One block's share of the table: slice `slice` of NS.  NT threads (a multiple of 32, <= 1024, dividing NB), all of
// which must call.  hostPlan: the plan made on the host (data-independent radius: a PREFIX of the paper's table, the
// search goes on beyond it by enumeration, nothing is needed from k_norm), or nullptr: radius_in >= 0 or, if < 0, the
// paper's radius from the control block (table_radius_from_ctl).
template <int NT, int ENT, int NB, int NS>
__device__ __forceinline__ void table_build_slice(TableSmem<ENT, NB, NS>& S, const GridP& g, const EvalP& e,
                                                  Ctl* __restrict__ ctl, const TablePlan* hostPlan, float radius_in,
                                                  long long cap, int4* __restrict__ table,
                                                  unsigned* __restrict__ tmpL, unsigned* __restrict__ tmpIdx, int slice)
{
    static_assert(NB % NT == 0 && NT % 32 == 0 && NT <= 1024 && NB % NS == 0, "thread count");
    constexpr int PER = NB / NT;
    constexpr int TAB_BUCKETS = NB, TAB_SLICE = NB / NS;
    const unsigned tid = threadIdx.x;

    if (tid == 0)
        S.plan = hostPlan ? *hostPlan
                          : table_plan_make(g, radius_in >= 0.0f ? radius_in : table_radius_from_ctl(g, e, ctl), cap, 0, NB);
    for (unsigned b = tid; b < TAB_BUCKETS; b += NT) S.start[b] = 0;
    __syncthreads();
    const TablePlan P = S.plan;
    const int bx = P.box[0], by = P.box[1], bz = P.box[2];
    const unsigned V = (unsigned)(bx * by * bz);
    const float R2 = P.R2, scale = P.scale;
    const unsigned mul0 = P.divMul[0], sh0 = P.divSh[0], mul1 = P.divMul[1], sh1 = P.divSh[1];
    auto bucket_of = [&](float L2) { return min(TAB_BUCKETS - 1, (int)(L2 * scale)); };
    auto cell_of = [&](unsigned i, int& mx, int& my, int& mz) {      // i = mx + bx * (my + by * mz), no division
        mz = (int)fast_div(i, mul1, sh1);
        const unsigned rem = i - (unsigned)mz * (unsigned)(bx * by);
        my = (int)fast_div(rem, mul0, sh0);
        mx = (int)(rem - (unsigned)my * (unsigned)bx);
    };

    // (1) histogram of the whole box (every block)
#pragma unroll 4
    for (unsigned i = tid; i < V; i += NT) {
        int mx, my, mz;
        cell_of(i, mx, my, mz);
        const float L2 = cell_L2(mx, my, mz, g);
        if (L2 < R2) atomicAdd(&S.start[bucket_of(L2)], 1u);
    }
    __syncthreads();
    // (2) exclusive scan of the 4096 bucket counts (PER per thread)
    {
        unsigned c[PER], s = 0;
#pragma unroll
        for (int j = 0; j < PER; ++j) { c[j] = S.start[tid * PER + j]; s += c[j]; }
        const unsigned lane = tid & 31u, warp = tid >> 5;
        unsigned incl = s;
#pragma unroll
        for (int k = 1; k < 32; k <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, incl, k);
            if (lane >= (unsigned)k) incl += t;
        }
        if (lane == 31) S.warpSums[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            unsigned w = lane < NT / 32 ? S.warpSums[lane] : 0u, wi = w;
#pragma unroll
            for (int k = 1; k < 32; k <<= 1) {
                const unsigned t = __shfl_up_sync(0xffffffffu, wi, k);
                if (lane >= (unsigned)k) wi += t;
            }
            S.warpSums[lane] = wi - w;
        }
        __syncthreads();
        unsigned run = S.warpSums[warp] + incl - s;
#pragma unroll
        for (int j = 0; j < PER; ++j) { S.start[tid * PER + j] = run; run += c[j]; }
        if (tid == NT - 1) S.start[TAB_BUCKETS] = run;
    }
    __syncthreads();
    const unsigned T = S.start[TAB_BUCKETS];
    // (3) this block's slice of buckets: collect its entries (order inside a bucket is arbitrary here)
    const int b0 = slice * TAB_SLICE;
    const unsigned lo0 = S.start[b0], cnt = S.start[b0 + TAB_SLICE] - lo0;
    const bool inSmem = cnt <= (unsigned)ENT;
    unsigned* const Ls = inSmem ? S.slice : tmpL + lo0;
    unsigned* const Is = inSmem ? S.slice + ENT : tmpIdx + lo0;
    for (unsigned b = tid; b < (unsigned)TAB_SLICE; b += NT) S.cursor[b] = S.start[b0 + b] - lo0;
    __syncthreads();
    if (cnt > 0) {
#pragma unroll 4
        for (unsigned i = tid; i < V; i += NT) {
            int mx, my, mz;
            cell_of(i, mx, my, mz);
            const float L2 = cell_L2(mx, my, mz, g);
            if (L2 < R2) {
                const int b = bucket_of(L2) - b0;
                if (b >= 0 && b < TAB_SLICE) {
                    const unsigned pos = atomicAdd(&S.cursor[b], 1u);
                    Ls[pos] = __float_as_uint(L2);
                    Is[pos] = i;
                }
            }
        }
    }
    __threadfence_block();
    __syncthreads();
    // (4) exact rank inside the bucket, write the final entry
    for (unsigned i = tid; i < cnt; i += NT) {
        const unsigned Lb = Ls[i], id = Is[i];
        const int b = bucket_of(__uint_as_float(Lb));
        const unsigned lo = S.start[b] - lo0, hi = S.start[b + 1] - lo0;
        unsigned rank = 0;
        for (unsigned j = lo; j < hi; ++j) {
            const unsigned Lj = Ls[j];
            rank += (Lj < Lb) || (Lj == Lb && Is[j] < id);
        }
        int mx, my, mz;
        cell_of(id, mx, my, mz);
        table[lo0 + lo + rank] = make_int4((int)Lb, mx, my, mz);
    }
    if (slice == 0 && tid == 0) {
        ctl->tableCount = T;
        ctl->tableTrunc = P.trunc;
        ctl->Rtab2 = R2;
        ctl->box[0] = bx; ctl->box[1] = by; ctl->box[2] = bz;
    }
    __syncthreads();                                     // the caller may reuse the shared memory
}

// Stand-alone builder: TAB_BLOCKS blocks of TAB_THREADS threads, TAB_DYN_SMEM bytes of dynamic shared memory.
__global__ void __launch_bounds__(TAB_THREADS)
k_offset_table(GridP g, EvalP e, Ctl* __restrict__ ctl, float radius_in, long long cap, int4* __restrict__ table,
               unsigned* __restrict__ tmpL, unsigned* __restrict__ tmpIdx, int prefix)
{
    using Smem = TableSmem<TAB_SMEM_ENTRIES, TAB_BUCKETS, TAB_BLOCKS>;
    extern __shared__ __align__(16) unsigned char tabRaw[];
    Smem& S = *reinterpret_cast<Smem*>(tabRaw);
    __shared__ TablePlan prefixPlan;
    if (prefix) {
        if (threadIdx.x == 0) prefixPlan = table_plan_make(g, radius_in, cap, 1, TAB_BUCKETS);
        __syncthreads();
    }
    table_build_slice<TAB_THREADS, TAB_SMEM_ENTRIES, TAB_BUCKETS, TAB_BLOCKS>(
        S, g, e, ctl, prefix ? &prefixPlan : nullptr, radius_in, cap, table, tmpL, tmpIdx, (int)blockIdx.x);
}

}  // namespace gamma_b200
