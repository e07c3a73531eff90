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
#include <math.h>

namespace beagle {

constexpr int kRankThreads = 256;
constexpr int kRankMaxSample = 1024;

__host__ __device__ __forceinline__ float rank_goodness(float f, int maximise)
{
    const float g = maximise ? f : -f;
#ifdef __CUDA_ARCH__
    return f != f ? __int_as_float(0xff800000) : g;                 // NaN: worse than every number (R24)
#else
    return f != f ? -INFINITY : g;                                  // (the host build of the same line: beagle_debug_rank, test only)
#endif
}

__global__ void __launch_bounds__(kRankThreads) k_rank(const float* __restrict__ fitness, long long P,
                                                       const long long* __restrict__ sample_idx, int n_sample, int maximise,
                                                       uint8_t* __restrict__ decile, unsigned long long* __restrict__ hist)
{
#define RK_SHARED(type, name, count) __shared__ type name[count];
#define RK_TID threadIdx.x
#define RK_BID blockIdx.x
#define RK_GDIM gridDim.x
#define RK_SYNC __syncthreads();
#define RK_LDG(p) __ldg(p)
#define RK_ATOMIC_ADD(p, v) atomicAdd(p, v)
#include "rank_body.inc"
#undef RK_SHARED
#undef RK_TID
#undef RK_BID
#undef RK_GDIM
#undef RK_SYNC
#undef RK_LDG
#undef RK_ATOMIC_ADD
}

} // namespace beagle
