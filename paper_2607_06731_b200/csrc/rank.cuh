// rank.cuh — Monte-Carlo ranking on the device (Table 2; D8).
//
// "Beagle takes a random sample of 100 individuals and uses those 100 individuals to estimate the population
// percentiles. Through one pass of the population then, individuals are assigned to their specific percentile"
// (P:106). The draw is the caller's (sample_idx), so the step is deterministic: every CTA gathers the sampled
// fitnesses, turns them into "goodness" (higher is better, NaN worst) and rank-sorts them in shared memory (100 x 100
// comparisons: cheaper than a second launch); then one grid-stride pass: for each individual a binary search counts
// the samples strictly worse, decile = min(9, 10 * worse / n_sample), one byte out, and a 10-bin histogram (from
// which the host sizes the next generation: expected births = sum hist[g] * Table2[g]).
// HBM-bound by construction: 4 bytes in, 1 byte out per individual.
#pragma once
#include <stdint.h>

namespace beagle {

constexpr int kRankThreads = 256;
constexpr int kRankMaxSample = 1024;

__device__ __forceinline__ float rank_goodness(float f, int maximise)
{
    const float g = maximise ? f : -f;
    return f != f ? __int_as_float(0xff800000) : g;                 // NaN: worse than every number (R24)
}

__global__ void __launch_bounds__(kRankThreads) k_rank(const float* __restrict__ fitness, long long P,
                                                       const long long* __restrict__ sample_idx, int n_sample, int maximise,
                                                       uint8_t* __restrict__ decile, unsigned long long* __restrict__ hist)
{
    __shared__ float raw[kRankMaxSample], srt[kRankMaxSample];
    __shared__ unsigned int h[10];
    if (threadIdx.x < 10) h[threadIdx.x] = 0;
    for (int j = threadIdx.x; j < n_sample; j += kRankThreads) raw[j] = rank_goodness(__ldg(fitness + sample_idx[j]), maximise);
    __syncthreads();
    for (int t = threadIdx.x; t < n_sample; t += kRankThreads) {    // rank sort, ties by index: a permutation
        const float v = raw[t];
        int r = 0;
        for (int j = 0; j < n_sample; ++j) { const float w = raw[j]; r += (w < v) || (w == v && j < t); }
        srt[r] = v;
    }
    __syncthreads();
    const long long stride = (long long)gridDim.x * kRankThreads;
    for (long long i = (long long)blockIdx.x * kRankThreads + threadIdx.x; i < P; i += stride) {
        const float g = rank_goodness(__ldg(fitness + i), maximise);
        int lo = 0, hi = n_sample;                                  // first position whose sample is not < g
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (srt[mid] < g) lo = mid + 1; else hi = mid; }
        int d = (10 * lo) / n_sample;
        d = d > 9 ? 9 : d;
        decile[i] = (uint8_t)d;
        atomicAdd(&h[d], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 10 && h[threadIdx.x]) atomicAdd(hist + threadIdx.x, (unsigned long long)h[threadIdx.x]);
}

} // namespace beagle
