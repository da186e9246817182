// common.cuh -- shared device-side definitions of libgamma_b200 (sm_100a).
// Notation follows the paper: D_r reference dose, D_e evaluation dose, dD dose criterion, DTA distance
// criterion, L the normalised spatial distance of the offset table (Algorithm A1).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace gamma_b200 {

// Geometry of the dose grid in units of the DTA criterion.  Passed to kernels by value.
struct GridP {
    int n[3];        // nx, ny, nz
    int stride[3];   // 1, nx, nx*ny
    int N;           // nx*ny*nz
    float h[3];      // spacing / DTA; 0 for a dropped axis (size 1)
    float hh[3];     // h^2
    float invA[8];   // invA[T] = 1 / sum_{a in T} h_a^2 over axis subsets T (bit0 x, bit1 y, bit2 z); 0 if T has a dropped axis
    float K3, K5, K6;          // h_a^2 h_b^2 / (h_a^2 + h_b^2) for the pairs xy, xz, yz
    float Kxy7, Kyz7, Kzx7;    // h_a^2 h_b^2 / (h_x^2 + h_y^2 + h_z^2)
    float rho_link2; // squared distance from a voxel to the boundary of its star (3D only), slightly shrunk
    float hmin2;     // squared smallest h over the active axes, slightly shrunk: nothing outside the 2^n cells
                     // that touch a voxel is closer than this
    int all_active;  // 1 when all three axes have size > 1
    unsigned divMul[2], divSh[2];  // exact division of lin < 2^31 by nx (0) and by nx*ny (1): see fast_div
};

// q = n / d for n < 2^31 with M = floor(2^(31+l) / d) + 1, l = ceil(log2 d) (set up on the host).
__device__ __forceinline__ unsigned fast_div(unsigned n, unsigned mul, unsigned sh)
{
    return (unsigned)(((unsigned long long)n * mul) >> sh);
}
__device__ __forceinline__ void voxel_coords(const GridP& g, int lin, int& ix, int& iy, int& iz)
{
    iz = (int)fast_div((unsigned)lin, g.divMul[1], g.divSh[1]);
    const int rem = lin - iz * g.stride[2];
    iy = (int)fast_div((unsigned)rem, g.divMul[0], g.divSh[0]);
    ix = rem - iy * g.n[0];
}

// Criteria (Eq. 1) and exclusion policy (readings 8-10).
struct EvalP {
    float DD;        // dose-difference criterion, fraction
    float cutoff;    // low-dose cutoff, fraction of D_norm
    float norm_dose; // D_norm if > 0, else taken from Ctl::normOrd
    int mode;        // 0 global, 1 local
    int algo;        // 0: closed form on owned faces (default); 1: grid vertices only (classical discrete gamma,
                     // comparator); 2: the six Kuhn tetrahedra of a cell by the negative-weight recursion (ju_simplex.cuh)
    unsigned call;   // number of the call on its workspace (device timeline, GAMMA_TRACE)
};

// Device control block: everything the pipeline decides on the device (no host sync on the path).
// Slots 0 .. CTL_ROT-1 rotate between the consecutive calls of a workspace, slot CTL_STANDALONE serves the stand-alone
// entry points, slot CTL_CAPTURE the calls captured into a caller's CUDA graph (cleared by a memset node).  Each slot
// has its own small offset table.  The invariant, in one place: k_norm of call i zeroes slot (i + 1) % CTL_ROT for
// call i + 1; that slot was last used by call i - 2, which has completed before k_norm(i) writes anything: k_norm(i)
// either waits for the operation in front of it before doing anything (default), or -- started early, in the tail of
// call i - 1 on a library-owned stream -- is launched only after k_star(i - 1) has completed, which is after
// k_classify(i - 1) passed its wait for k_norm(i - 1), whose last act is to wait for the end of call i - 2.
constexpr int CTL_ROT = 3, CTL_STANDALONE = 3, CTL_CAPTURE = 4, CTL_SLOTS = 5;
constexpr int KEY_DIGITS = 256;
struct Ctl {
    unsigned normOrd;      // max(ref) as an order-preserving uint
    unsigned maxAbsDD;     // bits of max |D_r - D_e| over all voxels (non-negative float): A1 step 1
    unsigned maxRatio;     // local mode: bits of max |D_r - D_e| / D_r over voxels with D_r > 0
    unsigned maxKeyBits;   // largest key of the search list (bits of a non-negative float), diagnostic
    unsigned nEval;        // M: evaluated voxels
    unsigned nSearch;      // voxels in the table-search work list
    unsigned workCounter;  // dynamic work fetch of the table search
    unsigned tileCounter;  // dynamic chunk fetch of the prep/star kernel
    unsigned tableCount;   // octant entries in the offset table
    unsigned tableTrunc;   // 1 if the table was cut at table_cap
    float Rtab2;           // squared radius the table covers
    int box[3];            // table box: m_a in [0, box_a)
    unsigned sortN;        // element count for gamma_sort_pairs
    unsigned nDeep;        // depth-class lists (presort 4): items in the deep list
    unsigned pad0_;
    float invGlobal;       // 1 / (DD * D_norm) rounded to fp32 (global criterion), written by k_classify
    unsigned long long visits;       // owner vertices evaluated by the table search
    unsigned zeros[32];              // always zero (ticket_one)
    unsigned hist[KEY_DIGITS];       // digit histogram of the search list (bucket presort)
    unsigned cursor[KEY_DIGITS];     // scatter cursors of the bucket presort
};

// ------------------------------------------------------------------------------------------------
// Device timeline (build with -DGAMMA_TRACE, e.g. GAMMA_NVCC_EXTRA=-DGAMMA_TRACE python -m paper_1012_1900_b200.build
// --force; read with gamma_trace_read / bench_suite.py --suite trace).  Every kernel of a call stamps %globaltimer when
// its first thread starts, when it passes its griddepcontrol.wait, and when its last block ends, into the record of the
// call (call number modulo TRACE_CALLS).  Without the macro nothing is compiled into the kernels.
// ------------------------------------------------------------------------------------------------
constexpr int TRACE_CALLS = 256;
constexpr int TRACE_KERNELS = 4;      // 0 k_norm, 1 k_classify, 2 k_star, 3 k_table_search
struct TraceRec {
    unsigned long long first, waited, last;   // ns: earliest start, latest "dependency met", latest block end
    unsigned long long pad_;
};
// Per-warp records of the LAST k_table_search launch (same build): when the warp started, passed the dependency wait,
// finished its first work unit and ended, and how many units it took.
constexpr int TRACE_WARPS = 8192;
struct TraceWarp { unsigned long long start, waited, firstUnit, end, units, pad_[3]; };
#ifdef GAMMA_TRACE
__device__ TraceWarp* g_trace_warps = nullptr;   // TRACE_WARPS records, set by the host
__device__ TraceRec* g_trace_buf = nullptr;   // TRACE_CALLS x TRACE_KERNELS records, set by the host
__device__ __forceinline__ unsigned long long trace_now()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void trace_first(unsigned call, int k)
{
    if (threadIdx.x == 0 && g_trace_buf) atomicMin(&g_trace_buf[(call % TRACE_CALLS) * TRACE_KERNELS + k].first, trace_now());
}
__device__ __forceinline__ void trace_waited(unsigned call, int k)
{
    if (threadIdx.x == 0 && g_trace_buf) atomicMax(&g_trace_buf[(call % TRACE_CALLS) * TRACE_KERNELS + k].waited, trace_now());
}
__device__ __forceinline__ void trace_last(unsigned call, int k)
{
    if (threadIdx.x == 0 && g_trace_buf) atomicMax(&g_trace_buf[(call % TRACE_CALLS) * TRACE_KERNELS + k].last, trace_now());
}
#else
__device__ __forceinline__ void trace_first(unsigned, int) {}
__device__ __forceinline__ void trace_waited(unsigned, int) {}
__device__ __forceinline__ void trace_last(unsigned, int) {}
#endif

__device__ __forceinline__ unsigned ticket_one(const Ctl* ctl) { return 1u + ctl->zeros[threadIdx.x & 31]; }

// Monotone 8-bit quantisation of a non-negative key: 32 steps per octave over [2^-3, 2^5), clamped.
// This is the digit of the one-pass MSD radix presort of the search work list.
__device__ __forceinline__ unsigned key_digit(float key)
{
    const int d = (int)(__float_as_uint(key) >> 18) - ((127 - 3) << 5);
    return (unsigned)min(max(d, 0), KEY_DIGITS - 1);
}

__host__ __device__ inline unsigned float_to_ordered(float f)
{
#if defined(__CUDA_ARCH__)
    unsigned b = __float_as_uint(f);
#else
    union { float f; unsigned u; } cv; cv.f = f; unsigned b = cv.u;
#endif
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__host__ __device__ inline float ordered_to_float(unsigned u)
{
    unsigned b = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u;
#if defined(__CUDA_ARCH__)
    return __uint_as_float(b);
#else
    union { float f; unsigned u; } cv; cv.u = b; return cv.f;
#endif
}

// squared normalised minimum spatial distance of the cell [o, o+1] with m_a = max(o_a, -o_a-1)
// (reading 4).  One definition for the table builder and the beyond-table enumeration.
__device__ __forceinline__ float cell_L2(int mx, int my, int mz, const GridP& g)
{
    const float ax = (float)mx * g.h[0], ay = (float)my * g.h[1], az = (float)mz * g.h[2];
    return fmaf(ax, ax, fmaf(ay, ay, az * az));
}

// Work ticket: a counter incremented by one whose old value is not needed before the end of the current work item.
// ptxas aggregates an integer atomicAdd (or PTX atom.add / atom.inc, 32 or 64 bit) with a warp-uniform addend over the
// active lanes -- vote, popc, the leader's ATOMG, SHFL of the result -- and that shuffle waits for the atomic right
// where it was issued (measured: the largest single stall of k_table_search, 19 % of its warp samples; fp32 atomics are
// not aggregated but serialise on one address: 5 us slower).  With an addend it cannot prove uniform (1 + a zero word
// loaded per lane from the control block) a partially active warp gets a plain ATOMG per lane, whose result is consumed
// where the program uses it.  Call from ONE lane of the warp with `one` = ticket_one(ctl).
__device__ __forceinline__ unsigned ticket_next(unsigned* p, unsigned one)
{
    unsigned r;
    asm volatile("atom.global.add.u32 %0, [%1], %2;" : "=r"(r) : "l"(p), "r"(one));
    return r;
}

__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}

}  // namespace gamma_b200
