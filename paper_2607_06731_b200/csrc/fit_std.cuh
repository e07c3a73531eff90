// fit_std.cuh — the Std integer-reward fitness family (Eq. 5 at P:503-506; D9):
// StdFitFunc and its Square / Cube / Hyper variants (power 1, 2, 3, 8). Per valid pair
//     M if max(|f|, |y|) = 0;   rint(M q^p - [f and y of opposite sign] M / 11)   with q = min(|f|,|y|) / max(|f|,|y|);
// a pair with exactly one side finite scores -M, with neither +M; the score is the sum over the cases.
// fp32, in the order the oracle states (the integer is decided in the paper's precision on both sides):
// |.|, min / max, one IEEE division, the power by squarings, * M, - M/11, round half to even.
// Rewards are integers, so the sum is exact in fp32 while |score| < 2^24 (M N <= 1.6e7) and its order does not matter;
// it is still taken in the fixed order of the other reductions.
#pragma once
#include <stdint.h>
#include <string.h>
#include <math.h>

// std_reward is compiled for the host too (beagle_debug_std_reward, test only: the integer a reward is rounded to is decided by fp32
// arithmetic, and a CPU test holds this function against the oracle's bit for bit). The device build is these intrinsics, unchanged;
// on the host the same IEEE single-precision operations written plainly (no contraction: mul and sub are separate statements and the
// host build has no fused multiply-add to contract them into).
#ifdef __CUDA_ARCH__
#define BGS_DIV(a, b) __fdiv_rn(a, b)
#define BGS_MUL(a, b) __fmul_rn(a, b)
#define BGS_SUB(a, b) __fsub_rn(a, b)
#define BGS_INF       __int_as_float(0x7f800000)
#define BGS_BITS(f)   __float_as_int(f)
#else
namespace beagle { inline int std_bits_host(float f) { int i; memcpy(&i, &f, 4); return i; } }
#define BGS_DIV(a, b) ((float)(a) / (float)(b))
#define BGS_MUL(a, b) ((float)(a) * (float)(b))
#define BGS_SUB(a, b) ((float)(a) - (float)(b))
#define BGS_INF       INFINITY
#define BGS_BITS(f)   beagle::std_bits_host(f)
#endif

namespace beagle {

// Straight-line (selects, no branches: the cases of a lane take the same path); the arithmetic and its order are the
// oracle's. yv: the target is finite (it does not change with the individual).
__host__ __device__ __forceinline__ float std_reward(float f, float y, float M, float pen, int power)
{
    const float a = fabsf(f), b = fabsf(y);
    const bool vf = a < BGS_INF, vy = b < BGS_INF;
    const float mx = fmaxf(a, b), mn = fminf(a, b);
    const float q = BGS_DIV(mn, mx);                         // 0/0, inf/inf: NaN, replaced below
    float qp = q;
    if (power == 2) qp = BGS_MUL(q, q);                      // warp-uniform
    else if (power == 3) qp = BGS_MUL(BGS_MUL(q, q), q);
    else if (power == 8) { qp = BGS_MUL(q, q); qp = BGS_MUL(qp, qp); qp = BGS_MUL(qp, qp); }
    const float t = BGS_MUL(M, qp);
    // opposite signs: both non-zero and the sign bits differ (decided on the signs, not on a product that may underflow)
    const bool opp = mn > 0.f && ((BGS_BITS(f) ^ BGS_BITS(y)) < 0);
    float r = rintf(opp ? BGS_SUB(t, pen) : t);
    r = mx == 0.f ? M : r;
    return (vf && vy) ? r : (vf != vy ? -M : M);
}

} // namespace beagle
