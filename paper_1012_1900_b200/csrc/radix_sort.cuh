// radix_sort.cuh -- hand-written LSD radix sort of (key, value) u32 pairs, element count on the device.
//
// Subsystem (3) of the gamma path: the voxel work list {voxel index, key} is sorted so that neighbouring
// lanes get similar search depth (Algorithm A2 step 3, used Thrust there).
// Keys are bit patterns of non-negative fp32 values, which order like unsigned integers.
//
// One pass per 8-bit digit, three kernels per pass, all reading the element count from device memory so
// that the pipeline never synchronises with the host:
//   k_radix_hist    per-tile digit histogram            -> tileHist[digit][tile]
//   k_radix_scan    exclusive scan in digit-major order -> global base of every (digit, tile)
//   k_radix_scatter stable ranking inside the tile (warp match + per-warp counters) and scatter
// Tile = 256 threads x 8 keys; a warp owns 256 consecutive keys and ranks them 32 at a time, which keeps
// the sort stable.  Algorithmic traffic per pass: read keys twice + values once, write both: 20 B/pair.
#pragma once
#include "common.cuh"

namespace gamma_b200 {

constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS = 8;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;  // 2048
constexpr int SORT_RADIX = 256;

__device__ __forceinline__ unsigned sort_num_tiles(unsigned n) { return (n + SORT_TILE - 1) / SORT_TILE; }

__global__ void __launch_bounds__(SORT_THREADS)
k_radix_hist(const unsigned* __restrict__ keys, const unsigned* __restrict__ nPtr, int shift,
             unsigned* __restrict__ tileHist)
{
    const unsigned n = *nPtr;
    const unsigned numTiles = sort_num_tiles(n);
    __shared__ unsigned hist[SORT_RADIX];
    for (unsigned tile = blockIdx.x; tile < numTiles; tile += gridDim.x) {
        hist[threadIdx.x] = 0;
        __syncthreads();
        const unsigned base = tile * SORT_TILE;
#pragma unroll
        for (int j = 0; j < SORT_ITEMS; ++j) {
            const unsigned i = base + j * SORT_THREADS + threadIdx.x;
            if (i < n) atomicAdd(&hist[(keys[i] >> shift) & 0xffu], 1u);
        }
        __syncthreads();
        tileHist[threadIdx.x * numTiles + tile] = hist[threadIdx.x];
        __syncthreads();
    }
}

// exclusive scan of tileHist[0 .. 256*numTiles) in place; one block of 1024 threads.
__global__ void __launch_bounds__(1024)
k_radix_scan(unsigned* __restrict__ tileHist, const unsigned* __restrict__ nPtr)
{
    const unsigned n = *nPtr;
    const unsigned total = sort_num_tiles(n) * SORT_RADIX;
    if (total == 0) return;
    const unsigned per = (total + 1023u) / 1024u;
    const unsigned lo = min(threadIdx.x * per, total), hi = min(lo + per, total);
    unsigned sum = 0;
    for (unsigned i = lo; i < hi; ++i) sum += tileHist[i];
    // block exclusive scan of the 1024 partial sums
    __shared__ unsigned warpSums[32];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned incl = sum;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, s);
        if (lane >= (unsigned)s) incl += t;
    }
    if (lane == 31) warpSums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        unsigned w = warpSums[lane], wi = w;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, wi, s);
            if (lane >= (unsigned)s) wi += t;
        }
        warpSums[lane] = wi - w;
    }
    __syncthreads();
    unsigned run = warpSums[warp] + incl - sum;
    for (unsigned i = lo; i < hi; ++i) {
        const unsigned t = tileHist[i];
        tileHist[i] = run;
        run += t;
    }
}

__global__ void __launch_bounds__(SORT_THREADS)
k_radix_scatter(const unsigned* __restrict__ keysIn, const unsigned* __restrict__ valsIn,
                unsigned* __restrict__ keysOut, unsigned* __restrict__ valsOut,
                const unsigned* __restrict__ nPtr, int shift, const unsigned* __restrict__ tileHist)
{
    const unsigned n = *nPtr;
    const unsigned numTiles = sort_num_tiles(n);
    constexpr int WARPS = SORT_THREADS / 32;
    __shared__ unsigned wc[WARPS][SORT_RADIX];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned ltMask = (1u << lane) - 1u;
    for (unsigned tile = blockIdx.x; tile < numTiles; tile += gridDim.x) {
#pragma unroll
        for (int w = 0; w < WARPS; ++w) wc[w][threadIdx.x] = 0;
        __syncthreads();
        unsigned key[SORT_ITEMS], rank[SORT_ITEMS];
        const unsigned base = tile * SORT_TILE + warp * (32 * SORT_ITEMS);
#pragma unroll
        for (int r = 0; r < SORT_ITEMS; ++r) {
            const unsigned i = base + r * 32 + lane;
            const bool valid = i < n;
            key[r] = valid ? keysIn[i] : 0xffffffffu;
            const unsigned digit = valid ? ((key[r] >> shift) & 0xffu) : 0x100u;
            const unsigned peers = __match_any_sync(0xffffffffu, digit);
            unsigned prev = 0;
            if (valid) prev = wc[warp][digit];
            __syncwarp();
            if (valid && (peers & ltMask) == 0) wc[warp][digit] = prev + __popc(peers);
            __syncwarp();
            rank[r] = prev + __popc(peers & ltMask);
        }
        __syncthreads();
        {   // thread d turns the per-warp counts of digit d into global base positions
            unsigned run = tileHist[threadIdx.x * numTiles + tile];
#pragma unroll
            for (int w = 0; w < WARPS; ++w) {
                const unsigned t = wc[w][threadIdx.x];
                wc[w][threadIdx.x] = run;
                run += t;
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < SORT_ITEMS; ++r) {
            const unsigned i = base + r * 32 + lane;
            if (i < n) {
                const unsigned pos = wc[warp][(key[r] >> shift) & 0xffu] + rank[r];
                keysOut[pos] = key[r];
                valsOut[pos] = valsIn[i];
            }
        }
        __syncthreads();
    }
}

// Enqueue the passes for key bits [beginBit, endBit).  Buffers ping-pong between (k0, v0) and (k1, v1);
// returns 0 if the sorted data ends in (k0, v0), 1 if in (k1, v1).  maxN bounds *nPtr (grid sizing only).
inline int radix_sort_enqueue(unsigned* k0, unsigned* v0, unsigned* k1, unsigned* v1, const unsigned* nPtr,
                              long long maxN, int beginBit, int endBit, unsigned* tileHist, cudaStream_t st)
{
    long long tiles = (maxN + SORT_TILE - 1) / SORT_TILE;
    int grid = (int)(tiles < 1 ? 1 : (tiles > 148 * 16 ? 148 * 16 : tiles));
    int cur = 0;
    for (int bit = beginBit; bit < endBit; bit += 8) {
        unsigned* ki = cur ? k1 : k0; unsigned* vi = cur ? v1 : v0;
        unsigned* ko = cur ? k0 : k1; unsigned* vo = cur ? v0 : v1;
        k_radix_hist<<<grid, SORT_THREADS, 0, st>>>(ki, nPtr, bit, tileHist);
        k_radix_scan<<<1, 1024, 0, st>>>(tileHist, nPtr);
        k_radix_scatter<<<grid, SORT_THREADS, 0, st>>>(ki, vi, ko, vo, nPtr, bit, tileHist);
        cur ^= 1;
    }
    return cur;
}

}  // namespace gamma_b200
