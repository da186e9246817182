// radix_sort.cuh -- hand-written LSD radix sort of (key, value) u32 pairs, element count on the device.
//
// Subsystem (3) of the gamma path: the voxel work list {voxel index, key} is sorted so that neighbouring
// lanes get similar search depth (Algorithm A2 step 3, used Thrust there).
// Keys are bit patterns of non-negative fp32 values, which order like unsigned integers.
//
// One pass per 8-bit digit, three kernels per pass, all reading the element count from device memory so
// that the pipeline never synchronises with the host:
//   k_radix_hist    per-tile digit histogram            -> tileHist[digit][tile]
//   k_radix_scan    exclusive scan along the tiles of every digit (one block per digit) + digit totals
//   k_radix_scatter stable ranking inside the tile (warp match + per-warp counters) and scatter
// Tile = 256 threads x 16 keys; a warp owns 512 consecutive keys and ranks them 32 at a time, which keeps
// the sort stable; the scatter stages the tile in shared memory in digit order before it stores it.  Algorithmic traffic per pass: read keys twice + values once, write both: 20 B/pair.
#pragma once
#include "common.cuh"

namespace gamma_b200 {

constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS = 16;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;  // 4096
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
        if (base + SORT_TILE <= n && (reinterpret_cast<uintptr_t>(keys) & 15u) == 0) {   // full tile: 16-byte loads
            const uint4* k4 = reinterpret_cast<const uint4*>(keys + base);
            uint4 v[SORT_ITEMS / 4];
#pragma unroll
            for (int j = 0; j < SORT_ITEMS / 4; ++j) v[j] = k4[j * SORT_THREADS + threadIdx.x];
#pragma unroll
            for (int j = 0; j < SORT_ITEMS / 4; ++j) {
                atomicAdd(&hist[(v[j].x >> shift) & 0xffu], 1u);
                atomicAdd(&hist[(v[j].y >> shift) & 0xffu], 1u);
                atomicAdd(&hist[(v[j].z >> shift) & 0xffu], 1u);
                atomicAdd(&hist[(v[j].w >> shift) & 0xffu], 1u);
            }
        } else {
#pragma unroll
            for (int j = 0; j < SORT_ITEMS; ++j) {
                const unsigned i = base + j * SORT_THREADS + threadIdx.x;
                if (i < n) atomicAdd(&hist[(keys[i] >> shift) & 0xffu], 1u);
            }
        }
        __syncthreads();
        tileHist[(size_t)threadIdx.x * numTiles + tile] = hist[threadIdx.x];
        __syncthreads();
    }
}

// Exclusive scan ALONG THE TILES of every digit's row tileHist[d][0 .. numTiles), in place, one block per digit
// (256 independent, coalesced scans instead of one scan over 256 * numTiles values: the single-block version of round 1
// took 3.5 ms of a 3.8 ms pass at 2^24 pairs, profiles/r2_sort.md); the row's total goes to digitTotal[d], from which
// every scatter block derives the digit's global base.
__global__ void __launch_bounds__(SORT_THREADS)
k_radix_scan(unsigned* __restrict__ tileHist, const unsigned* __restrict__ nPtr, unsigned* __restrict__ digitTotal)
{
    const unsigned numTiles = sort_num_tiles(*nPtr);
    unsigned* row = tileHist + (size_t)blockIdx.x * numTiles;
    __shared__ unsigned warpSums[SORT_THREADS / 32];
    __shared__ unsigned carry;
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (unsigned base = 0; base < numTiles; base += SORT_THREADS) {
        const unsigned i = base + threadIdx.x;
        const unsigned v = i < numTiles ? row[i] : 0u;
        unsigned incl = v;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, incl, s);
            if (lane >= (unsigned)s) incl += t;
        }
        if (lane == 31) warpSums[warp] = incl;
        __syncthreads();
        unsigned off = carry;
#pragma unroll
        for (int w = 0; w < SORT_THREADS / 32; ++w) off += (unsigned)w < warp ? warpSums[w] : 0u;
        if (i < numTiles) row[i] = off + incl - v;
        __syncthreads();
        if (threadIdx.x == SORT_THREADS - 1) carry = off + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) digitTotal[blockIdx.x] = carry;
}

// Scatter of one tile.  Ranking: a warp owns SORT_ITEMS x 32 consecutive keys and ranks them 32 at a time (warp match +
// per-warp digit counters), which keeps the sort stable.  The pairs are then STAGED in shared memory in digit order and
// written out from there: consecutive threads store consecutive positions of a digit's run, so a tile's 4 096 pairs leave
// as 256 runs of 16 pairs on average (full 32-byte sectors) instead of 4 096 single 4-byte stores whose partial sectors
// the memory system has to read back and merge (profiles/r2_sort.md).
#ifndef GAMMA_SORT_SCATTER_BLOCKS
#define GAMMA_SORT_SCATTER_BLOCKS 4
#endif
__global__ void __launch_bounds__(SORT_THREADS, GAMMA_SORT_SCATTER_BLOCKS)
k_radix_scatter(const unsigned* __restrict__ keysIn, const unsigned* __restrict__ valsIn,
                unsigned* __restrict__ keysOut, unsigned* __restrict__ valsOut,
                const unsigned* __restrict__ nPtr, int shift, const unsigned* __restrict__ tileHist,
                const unsigned* __restrict__ digitTotal)
{
    const unsigned n = *nPtr;
    const unsigned numTiles = sort_num_tiles(n);
    constexpr int WARPS = SORT_THREADS / 32;
    __shared__ unsigned wc[WARPS][SORT_RADIX];      // per-warp digit counts, then the warp's first local slot of the digit
    __shared__ unsigned digitBase[SORT_RADIX];      // global base of the digit (all tiles)
    __shared__ int toGlobal[SORT_RADIX];            // global position = local slot + toGlobal[digit]
    __shared__ unsigned scanWarp[WARPS];
    __shared__ unsigned sKey[SORT_TILE], sVal[SORT_TILE];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned ltMask = (1u << lane) - 1u;
    // exclusive scan over the 256 digits, one value per thread
    auto scan256 = [&](unsigned v) -> unsigned {
        unsigned incl = v;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, incl, s);
            if (lane >= (unsigned)s) incl += t;
        }
        if (lane == 31) scanWarp[warp] = incl;
        __syncthreads();
        unsigned off = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) off += (unsigned)w < warp ? scanWarp[w] : 0u;
        __syncthreads();
        return off + incl - v;
    };
    digitBase[threadIdx.x] = scan256(digitTotal[threadIdx.x]);
    for (unsigned tile = blockIdx.x; tile < numTiles; tile += gridDim.x) {
#pragma unroll
        for (int w = 0; w < WARPS; ++w) wc[w][threadIdx.x] = 0;
        __syncthreads();
        unsigned key[SORT_ITEMS], rank[SORT_ITEMS];
        const unsigned base = tile * SORT_TILE + warp * (32 * SORT_ITEMS);
        const unsigned tileCount = min((unsigned)SORT_TILE, n - tile * SORT_TILE);
#pragma unroll
        for (int r = 0; r < SORT_ITEMS; ++r) {
            const unsigned i = base + r * 32 + lane;
            const bool valid = i < n;
            key[r] = valid ? keysIn[i] : 0xffffffffu;
        }
#pragma unroll
        for (int r = 0; r < SORT_ITEMS; ++r) {
            const bool valid = base + r * 32 + lane < n;
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
        {   // thread d: the digit's count in the tile, its first local slot (scan over the digits), the warps' first slots
            unsigned cnt = 0;
#pragma unroll
            for (int w = 0; w < WARPS; ++w) cnt += wc[w][threadIdx.x];
            const unsigned start = scan256(cnt);
            unsigned run = start;
#pragma unroll
            for (int w = 0; w < WARPS; ++w) {
                const unsigned t = wc[w][threadIdx.x];
                wc[w][threadIdx.x] = run;
                run += t;
            }
            toGlobal[threadIdx.x] = (int)(digitBase[threadIdx.x] + tileHist[(size_t)threadIdx.x * numTiles + tile]) - (int)start;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < SORT_ITEMS; ++r) {
            if (base + r * 32 + lane < n) {
                const unsigned slot = wc[warp][(key[r] >> shift) & 0xffu] + rank[r];
                sKey[slot] = key[r];
                sVal[slot] = valsIn[base + r * 32 + lane];       // fetched here: 16 registers less while ranking
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < SORT_ITEMS; ++r) {
            const unsigned slot = r * SORT_THREADS + threadIdx.x;
            if (slot < tileCount) {
                const unsigned k = sKey[slot];
                const unsigned pos = (unsigned)((int)slot + toGlobal[(k >> shift) & 0xffu]);
                keysOut[pos] = k;
                valsOut[pos] = sVal[slot];
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
        unsigned* digitTotal = tileHist + (size_t)tiles * SORT_RADIX;     // 256 words behind the tile histograms
        k_radix_hist<<<grid, SORT_THREADS, 0, st>>>(ki, nPtr, bit, tileHist);
        k_radix_scan<<<SORT_RADIX, SORT_THREADS, 0, st>>>(tileHist, nPtr, digitTotal);
        k_radix_scatter<<<grid, SORT_THREADS, 0, st>>>(ki, vi, ko, vo, nPtr, bit, tileHist, digitTotal);
        cur ^= 1;
    }
    return cur;
}

}  // namespace gamma_b200
