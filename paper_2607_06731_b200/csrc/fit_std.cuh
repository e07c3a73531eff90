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

namespace beagle {

// Straight-line (selects, no branches: the cases of a lane take the same path); the arithmetic and its order are the
// oracle's. yv: the target is finite (it does not change with the individual).
__device__ __forceinline__ float std_reward(float f, float y, float M, float pen, int power)
{
    const float a = fabsf(f), b = fabsf(y);
    const bool vf = a < __int_as_float(0x7f800000), vy = b < __int_as_float(0x7f800000);
    const float mx = fmaxf(a, b), mn = fminf(a, b);
    const float q = __fdiv_rn(mn, mx);                       // 0/0, inf/inf: NaN, replaced below
    float qp = q;
    if (power == 2) qp = __fmul_rn(q, q);                    // warp-uniform
    else if (power == 3) qp = __fmul_rn(__fmul_rn(q, q), q);
    else if (power == 8) { qp = __fmul_rn(q, q); qp = __fmul_rn(qp, qp); qp = __fmul_rn(qp, qp); }
    const float t = __fmul_rn(M, qp);
    // opposite signs: both non-zero and the sign bits differ (decided on the signs, not on a product that may underflow)
    const bool opp = mn > 0.f && ((__float_as_int(f) ^ __float_as_int(y)) < 0);
    float r = rintf(opp ? __fsub_rn(t, pen) : t);
    r = mx == 0.f ? M : r;
    return (vf && vy) ? r : (vf != vy ? -M : M);
}

} // namespace beagle
