// fit_corr.cuh — the correlation fitness (Eq. 1-2; D7) as a warp-level
// reduction over the 16-cases-per-lane layout of both evaluation kernels (k_eval and k_eval_blockwise call the same
// functions on the same layout, so their results are bit-identical).
//
//   valid pair: f_i and y_i both finite; c1 = pairs with exactly one side finite; c2 = N - valid - c1;
//   r^2 = (Sfy / Sff) (Sfy / Syy) over the valid pairs, 0 when fewer than two are left or a variance is zero;
//   fitness = M r^4 valid - M (c1 - c2) - tax L.
//
// One pass (512 cases) is a two-pass summation in registers: values are first shifted by the first valid
// pair of the pass (so that constant data gives exactly zero variance), their means taken, then the centred
// sums. A second pass (N > 512) is merged with the pairwise update of the centred sums (Chan et al.):
//   S = S_a + S_b + (m_b - m_a)^2 n_a n_b / (n_a + n_b).
// Every sum is a per-lane chain over k = 0..15 followed by the 5-level butterfly: fixed order, reproducible.
#pragma once
#include <stdint.h>

namespace beagle {

struct CorrState { float n, mf, my, Sff, Syy, Sfy; int c1; };     // warp-uniform

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v = __fadd_rn(v, __shfl_xor_sync(0xffffffffu, v, m));
    return v;
}

__device__ __forceinline__ bool finite32(float v) { return fabsf(v) < __int_as_float(0x7f800000); }

// f[k], y[k]: case c0 + (k / 4) * 128 + lane * 4 + (k % 4); cases >= n do not count
__device__ __forceinline__ void corr_pass(const float (&f)[16], const float (&y)[16], int c0, int n, int lane, CorrState& st)
{
    uint32_t vmask = 0;
    int c1l = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const bool in = c0 + (k >> 2) * 128 + lane * 4 + (k & 3) < n;
        const bool vf = finite32(f[k]), vy = finite32(y[k]);
        if (in && vf && vy) vmask |= 1u << k;
        if (in && vf != vy) ++c1l;
    }
    int pack = __popc(vmask) | (c1l << 16);
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) pack += __shfl_xor_sync(0xffffffffu, pack, m);
    st.c1 += pack >> 16;
    const int nvp = pack & 0xffff;
    if (nvp == 0) return;                                          // warp-uniform
    // shift: the first valid pair of the pass
    float kf = 0.f, ky = 0.f;
#pragma unroll
    for (int k = 15; k >= 0; --k) if ((vmask >> k) & 1u) { kf = f[k]; ky = y[k]; }
    const int first = __ffs(__ballot_sync(0xffffffffu, vmask != 0)) - 1;
    kf = __shfl_sync(0xffffffffu, kf, first);
    ky = __shfl_sync(0xffffffffu, ky, first);
    float sf = 0.f, sy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) if ((vmask >> k) & 1u) { sf = __fadd_rn(sf, __fsub_rn(f[k], kf)); sy = __fadd_rn(sy, __fsub_rn(y[k], ky)); }
    const float np_ = (float)nvp;
    const float gf = __fdiv_rn(warp_sum(sf), np_), gy = __fdiv_rn(warp_sum(sy), np_);
    float sff = 0.f, syy = 0.f, sfy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) if ((vmask >> k) & 1u) {
        const float df = __fsub_rn(__fsub_rn(f[k], kf), gf), dy = __fsub_rn(__fsub_rn(y[k], ky), gy);
        sff = __fmaf_rn(df, df, sff); syy = __fmaf_rn(dy, dy, syy); sfy = __fmaf_rn(df, dy, sfy);
    }
    sff = warp_sum(sff); syy = warp_sum(syy); sfy = warp_sum(sfy);
    const float mfp = __fadd_rn(kf, gf), myp = __fadd_rn(ky, gy);
    if (st.n == 0.f) { st.n = np_; st.mf = mfp; st.my = myp; st.Sff = sff; st.Syy = syy; st.Sfy = sfy; return; }
    const float nt = __fadd_rn(st.n, np_), w = __fdiv_rn(__fmul_rn(st.n, np_), nt);
    const float ef = __fsub_rn(mfp, st.mf), ey = __fsub_rn(myp, st.my);
    st.Sff = __fadd_rn(__fadd_rn(st.Sff, sff), __fmul_rn(__fmul_rn(ef, ef), w));
    st.Syy = __fadd_rn(__fadd_rn(st.Syy, syy), __fmul_rn(__fmul_rn(ey, ey), w));
    st.Sfy = __fadd_rn(__fadd_rn(st.Sfy, sfy), __fmul_rn(__fmul_rn(ef, ey), w));
    st.mf = __fadd_rn(st.mf, __fmul_rn(ef, __fdiv_rn(np_, nt)));
    st.my = __fadd_rn(st.my, __fmul_rn(ey, __fdiv_rn(np_, nt)));
    st.n = nt;
}

__device__ __forceinline__ float corr_finish(const CorrState& st, int n, int len, float M, float tax)
{
    float r2 = 0.f;
    if (st.n >= 2.f && st.Sff > 0.f && st.Syy > 0.f) r2 = __fmul_rn(__fdiv_rn(st.Sfy, st.Sff), __fdiv_rn(st.Sfy, st.Syy));   // no overflow of Sff * Syy
    const int c2 = n - (int)st.n - st.c1;
    const float score = __fsub_rn(__fmul_rn(__fmul_rn(M, __fmul_rn(r2, r2)), st.n), __fmul_rn(M, (float)(st.c1 - c2)));
    return __fmaf_rn(-tax, (float)len, score);
}

} // namespace beagle
