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

__device__ __forceinline__ float std_reward(float f, float y, float M, float pen, int power)
{
    const bool vf = fabsf(f) < __int_as_float(0x7f800000), vy = fabsf(y) < __int_as_float(0x7f800000);
    if (!(vf && vy)) return vf != vy ? -M : M;
    const float a = fabsf(f), b = fabsf(y);
    const float mx = fmaxf(a, b), mn = fminf(a, b);
    if (mx == 0.f) return M;
    const float q = __fdiv_rn(mn, mx);
    float qp = q;
    if (power == 2) qp = __fmul_rn(q, q);
    else if (power == 3) qp = __fmul_rn(__fmul_rn(q, q), q);
    else if (power == 8) { qp = __fmul_rn(q, q); qp = __fmul_rn(qp, qp); qp = __fmul_rn(qp, qp); }
    float t = __fmul_rn(M, qp);
    if ((f < 0.f && y > 0.f) || (f > 0.f && y < 0.f)) t = __fsub_rn(t, pen);
    return rintf(t);
}

} // namespace beagle
