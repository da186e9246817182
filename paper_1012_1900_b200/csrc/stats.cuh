// stats.cuh -- subsystem (5): pass rate / gamma histogram reduction (BASELINE.json north_star (5); the
// paper reports no such step).  sum gamma^3 is the paper's work predictor.
// One read of gamma[n] (4 B per voxel): HBM/L2-bound; counts are integers, sums are fp64.
#pragma once
#include "common.cuh"
#include "../../include/gamma_b200.h"

namespace gamma_b200 {

constexpr int STATS_THREADS = 256;
constexpr int STATS_MAX_BINS = 4096;

__global__ void k_stats_clear(unsigned long long* __restrict__ hist, int nbins, gamma_summary* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nbins) hist[i] = 0ull;
    if (i == 0) {
        out->n_eval = 0; out->n_pass = 0; out->sum_gamma = 0.0; out->sum_gamma3 = 0.0;
        out->max_gamma = 0.0f; out->n_nan = 0; out->pad_ = 0;
    }
}

// One pass over gamma: float4 loads, per-thread counters, a shared-memory histogram (one private copy per warp when
// nbins <= STATS_WARP_BINS, so that the few populated bins are not hammered by all 256 threads), block reduction, then
// ONE set of global atomics per block.  Launched with programmatic dependent launch behind k_stats_clear: everything
// up to the global atomics runs while the clear drains.
constexpr int STATS_WARP_BINS = 128;
constexpr int STATS_WARPS = STATS_THREADS / 32;

__global__ void __launch_bounds__(STATS_THREADS)
k_stats(const float* __restrict__ gam, long long n, int nbins, float binScale,
        unsigned long long* __restrict__ hist, gamma_summary* __restrict__ out)
{
    extern __shared__ unsigned sHist[];                    // nbins * (private ? STATS_WARPS : 1)
    __shared__ unsigned sCnt[STATS_WARPS][3];
    __shared__ double sSum[STATS_WARPS][2];
    __shared__ float sMax[STATS_WARPS];
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const bool priv = nbins <= STATS_WARP_BINS;
    const int copies = priv ? STATS_WARPS : 1;
    for (int b = threadIdx.x; b < nbins * copies; b += blockDim.x) sHist[b] = 0;
    __syncthreads();
    unsigned* myHist = sHist + (priv ? (threadIdx.x >> 5) * nbins : 0);
    unsigned nEval = 0, nPass = 0, nNan = 0;
    double s1 = 0.0, s3 = 0.0;
    float mx = 0.0f;
    auto one = [&](float v) {
        if (v == v) {
            ++nEval;
            nPass += v <= 1.0f;
            const double dv = (double)v;
            s1 += dv;
            s3 += dv * dv * dv;
            mx = fmaxf(mx, v);
            const float fb = v * binScale;
            const int b = fb >= (float)(nbins - 1) ? nbins - 1 : (fb > 0.0f ? (int)fb : 0);
            atomicAdd(&myHist[b], 1u);
        } else {
            ++nNan;
        }
    };
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    if ((reinterpret_cast<uintptr_t>(gam) & 15u) == 0) {
        const float4* g4 = reinterpret_cast<const float4*>(gam);
        const long long n4 = n >> 2;
        for (long long i = tid; i < n4; i += stride) {
            const float4 v = __ldg(g4 + i);
            one(v.x); one(v.y); one(v.z); one(v.w);
        }
        for (long long i = (n4 << 2) + tid; i < n; i += stride) one(__ldg(gam + i));
    } else {
        for (long long i = tid; i < n; i += stride) one(__ldg(gam + i));
    }
    // warp, then block reduction (fixed order inside the block)
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        nEval += __shfl_xor_sync(0xffffffffu, nEval, s);
        nPass += __shfl_xor_sync(0xffffffffu, nPass, s);
        nNan += __shfl_xor_sync(0xffffffffu, nNan, s);
        s1 += __shfl_xor_sync(0xffffffffu, s1, s);
        s3 += __shfl_xor_sync(0xffffffffu, s3, s);
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    const int warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
        sCnt[warp][0] = nEval; sCnt[warp][1] = nPass; sCnt[warp][2] = nNan;
        sSum[warp][0] = s1; sSum[warp][1] = s3;
        sMax[warp] = mx;
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");    // hist / out are cleared from here on
    if (threadIdx.x == 0) {
        unsigned long long cE = 0, cP = 0;
        unsigned cN = 0;
        double a1 = 0.0, a3 = 0.0;
        float m = 0.0f;
        for (int w = 0; w < STATS_WARPS; ++w) {
            cE += sCnt[w][0]; cP += sCnt[w][1]; cN += sCnt[w][2];
            a1 += sSum[w][0]; a3 += sSum[w][1];
            m = fmaxf(m, sMax[w]);
        }
        if (cE) atomicAdd(&out->n_eval, cE);
        if (cP) atomicAdd(&out->n_pass, cP);
        if (cN) atomicAdd(&out->n_nan, cN);
        if (cE) {
            atomicAdd(&out->sum_gamma, a1);
            atomicAdd(&out->sum_gamma3, a3);
            atomicMax(reinterpret_cast<unsigned*>(&out->max_gamma), __float_as_uint(m));  // m >= 0
        }
    }
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) {
        unsigned c = 0;
        for (int w = 0; w < copies; ++w) c += sHist[w * nbins + b];
        if (c) atomicAdd(&hist[b], (unsigned long long)c);
    }
}

// ------------------------------------------------------------------------------------------------
// a6 fused into the gamma kernels (gamma_opts::stats_*): gamma is in a register when k_star / k_table_search write it,
// so the reduction costs a few shared-memory updates per voxel instead of a second pass over gamma[N].
// Every thread owns one slot in shared memory (no registers are held across the search), the histogram is a block-wide
// shared array; a block flushes once, at its end.  The caller's hist / summary are zeroed by k_norm, the first kernel
// of the call, which completes before any other kernel of the call starts.
// ------------------------------------------------------------------------------------------------
constexpr int FUSED_MAX_BINS = 1024;

struct StatsP {
    unsigned long long* hist;   // DEVICE, nbins u64; nullptr = no fused statistics
    gamma_summary* summary;     // DEVICE
    int nbins;
    float binScale;             // nbins / hist_max
};

struct StatSlot {
    double s1, s3;
    unsigned nEval, nPass;
    float mx;
    unsigned pad_;
};

template <int THREADS>
struct FusedStats {
    StatSlot slot[THREADS];
    unsigned hist[FUSED_MAX_BINS];
    double wSum[THREADS / 32][2];
    unsigned wCnt[THREADS / 32][2];
    float wMax[THREADS / 32];
};

// all threads of the block must call (contains a barrier when statistics are on)
template <int THREADS>
__device__ __forceinline__ void fused_stats_init(FusedStats<THREADS>& S, const StatsP& st)
{
    if (!st.hist) return;
    StatSlot z;
    z.s1 = 0.0; z.s3 = 0.0; z.nEval = 0; z.nPass = 0; z.mx = 0.0f; z.pad_ = 0;
    S.slot[threadIdx.x] = z;
    for (int b = threadIdx.x; b < st.nbins; b += THREADS) S.hist[b] = 0;
    __syncthreads();                                     // st.hist is uniform over the block
}

// one finite gamma value written by this thread (same bin rule as k_stats: decided in fp32)
template <int THREADS>
__device__ __forceinline__ void fused_stats_add(FusedStats<THREADS>& S, const StatsP& st, float v)
{
    if (!st.hist) return;
    if (!(v == v)) { atomicAdd(&st.summary->n_nan, 1u); return; }   // non-finite neighbourhood: counted as excluded
    StatSlot& z = S.slot[threadIdx.x];
    const double dv = (double)v;
    z.s1 += dv;
    z.s3 += dv * dv * dv;
    z.nEval += 1u;
    z.nPass += v <= 1.0f ? 1u : 0u;
    z.mx = fmaxf(z.mx, v);
    const float fb = v * st.binScale;
    const int b = fb >= (float)(st.nbins - 1) ? st.nbins - 1 : (fb > 0.0f ? (int)fb : 0);
    atomicAdd(&S.hist[b], 1u);
}

// block-wide flush: all threads of the block must call (contains __syncthreads)
template <int THREADS>
__device__ __forceinline__ void fused_stats_flush(FusedStats<THREADS>& S, const StatsP& st)
{
    if (!st.hist) return;
    __syncthreads();
    StatSlot z = S.slot[threadIdx.x];
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        z.s1 += __shfl_xor_sync(0xffffffffu, z.s1, s);
        z.s3 += __shfl_xor_sync(0xffffffffu, z.s3, s);
        z.nEval += __shfl_xor_sync(0xffffffffu, z.nEval, s);
        z.nPass += __shfl_xor_sync(0xffffffffu, z.nPass, s);
        z.mx = fmaxf(z.mx, __shfl_xor_sync(0xffffffffu, z.mx, s));
    }
    const int warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
        S.wSum[warp][0] = z.s1; S.wSum[warp][1] = z.s3;
        S.wCnt[warp][0] = z.nEval; S.wCnt[warp][1] = z.nPass;
        S.wMax[warp] = z.mx;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long cE = 0, cP = 0;
        double a1 = 0.0, a3 = 0.0;
        float m = 0.0f;
        for (int w = 0; w < THREADS / 32; ++w) {
            cE += S.wCnt[w][0]; cP += S.wCnt[w][1];
            a1 += S.wSum[w][0]; a3 += S.wSum[w][1];
            m = fmaxf(m, S.wMax[w]);
        }
        if (cE) {
            atomicAdd(&st.summary->n_eval, cE);
            atomicAdd(&st.summary->sum_gamma, a1);
            atomicAdd(&st.summary->sum_gamma3, a3);
            atomicMax(reinterpret_cast<unsigned*>(&st.summary->max_gamma), __float_as_uint(m));   // m >= 0
        }
        if (cP) atomicAdd(&st.summary->n_pass, cP);
    }
    for (int b = threadIdx.x; b < st.nbins; b += THREADS) {
        const unsigned c = S.hist[b];
        if (c) atomicAdd(&st.hist[b], (unsigned long long)c);
    }
}

// ------------------------------------------------------------------------------------------------
// FP32 ALU rate probe: 16 independent FFMA chains per thread (the "alu" roofline denominator).  The loop over
// PROBE_ITERS is unrolled 16 times: 256 FFMAs per trip against 3 loop instructions, so loop overhead is about 1 %.
// ------------------------------------------------------------------------------------------------
constexpr int PROBE_ITERS = 2048;
constexpr int PROBE_CHAINS = 16;

__global__ void __launch_bounds__(256) k_fp32_probe(float* __restrict__ sink, float a, float b)
{
    float x[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
#pragma unroll 16
    for (int it = 0; it < PROBE_ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < PROBE_CHAINS; ++c) x[c] = fmaf(x[c], a, b);
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) s += x[c];
    if (s == 123.456f) sink[0] = s;   // never true in practice; keeps the chains alive
}

}  // namespace gamma_b200
