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

__global__ void __launch_bounds__(STATS_THREADS)
k_stats(const float* __restrict__ gam, long long n, int nbins, float binScale,
        unsigned long long* __restrict__ hist, gamma_summary* __restrict__ out)
{
    extern __shared__ unsigned sHist[];
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) sHist[b] = 0;
    __syncthreads();
    unsigned nEval = 0, nPass = 0, nNan = 0;
    double s1 = 0.0, s3 = 0.0;
    float mx = 0.0f;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float v = __ldg(gam + i);
        if (v == v) {
            ++nEval;
            nPass += v <= 1.0f;
            const double dv = (double)v;
            s1 += dv;
            s3 += dv * dv * dv;
            mx = fmaxf(mx, v);
            const float fb = v * binScale;
            const int b = fb >= (float)(nbins - 1) ? nbins - 1 : (fb > 0.0f ? (int)fb : 0);
            atomicAdd(&sHist[b], 1u);
        } else {
            ++nNan;
        }
    }
    // block reduction
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        nEval += __shfl_xor_sync(0xffffffffu, nEval, s);
        nPass += __shfl_xor_sync(0xffffffffu, nPass, s);
        nNan += __shfl_xor_sync(0xffffffffu, nNan, s);
        s1 += __shfl_xor_sync(0xffffffffu, s1, s);
        s3 += __shfl_xor_sync(0xffffffffu, s3, s);
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, s));
    }
    if ((threadIdx.x & 31) == 0) {
        if (nEval) atomicAdd(&out->n_eval, (unsigned long long)nEval);
        if (nPass) atomicAdd(&out->n_pass, (unsigned long long)nPass);
        if (nNan) atomicAdd(&out->n_nan, nNan);
        if (nEval) {
            atomicAdd(&out->sum_gamma, s1);
            atomicAdd(&out->sum_gamma3, s3);
            atomicMax(reinterpret_cast<unsigned*>(&out->max_gamma), __float_as_uint(mx));  // mx >= 0
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += blockDim.x)
        if (sHist[b]) atomicAdd(&hist[b], (unsigned long long)sHist[b]);
}

// ------------------------------------------------------------------------------------------------
// FP32 ALU rate probe: 16 independent FFMA chains per thread (the "alu" roofline denominator).
// ------------------------------------------------------------------------------------------------
constexpr int PROBE_ITERS = 2048;
constexpr int PROBE_CHAINS = 16;

__global__ void __launch_bounds__(256) k_fp32_probe(float* __restrict__ sink, float a, float b)
{
    float x[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
#pragma unroll 1
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
