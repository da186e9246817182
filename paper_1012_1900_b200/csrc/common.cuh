// common.cuh -- shared device-side definitions of libgamma_b200 (sm_100a).
// Notation follows the paper: D_r reference dose, D_e evaluation dose, dD dose criterion, DTA distance
// criterion, L the normalised spatial distance of the offset table (Algorithm A1).
#pragma once
#include <cuda_runtime.h>
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
};

// Device control block: everything the pipeline decides on the device (no host sync on the path).
// One block per call SET.  CTL_ROT sets rotate between consecutive calls of a workspace (call number k uses set
// k % CTL_ROT: its own control block, offset table and work lists), one more serves the stand-alone entry points and
// one the calls captured into a caller's CUDA graph.  The invariant that makes calls in flight safe, in one place:
//   * a block is all zero whenever no call that uses it is in flight: the LAST block of a call's last kernel
//     (k_table_search) copies it to the set's report block (gamma_get_counters), zeroes it, and only then publishes
//     the call as done (SeqP::done = k + 1);
//   * calls are published in call order (that last block first waits for done == k), so "the last kernel of call k
//     has completed" implies "every earlier call has completed": stream order as the caller sees it is kept;
//   * the first kernel of call k (k_norm) does not write its block before done >= k + 1 - CTL_ROT, i.e. before the
//     previous user of the set has been published, and nothing else of call k starts before k_norm has completed.
constexpr int CTL_ROT = 4, CTL_STANDALONE = 4, CTL_CAPTURE = 5, CTL_SLOTS = 6;
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
    unsigned blocksDone;   // blocks of the call's last kernel that have finished (the last one publishes the call)
    float invGlobal;       // 1 / (DD * D_norm) rounded to fp32 (global criterion), written by k_classify
    unsigned long long visits;       // owner vertices evaluated by the table search
    unsigned hist[KEY_DIGITS];       // digit histogram of the search list (bucket presort)
    unsigned cursor[KEY_DIGITS];     // scatter cursors of the bucket presort
};

// Sequencing of the calls of one workspace (one word per workspace, never cleared by the kernels).
struct SeqP {
    unsigned* done;   // device word: number of calls published so far; nullptr = this call is not sequenced
    unsigned seq;     // this call's number k
    unsigned need;    // k_norm writes its control block only when done >= need (signed 32-bit difference)
};

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

__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, s));
    return v;
}

}  // namespace gamma_b200
