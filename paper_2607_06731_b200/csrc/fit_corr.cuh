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

// merge the centred sums of one pass (np_ valid pairs, means mfp, myp) into the running state
__device__ __forceinline__ void corr_merge(CorrState& st, float np_, float mfp, float myp, float sff, float syy, float sfy)
{
    if (__all_sync(0xffffffffu, st.n == 0.f)) { st.n = np_; st.mf = mfp; st.my = myp; st.Sff = sff; st.Syy = syy; st.Sfy = sfy; return; }
    const float nt = __fadd_rn(st.n, np_), w = __fdiv_rn(__fmul_rn(st.n, np_), nt);
    const float ef = __fsub_rn(mfp, st.mf), ey = __fsub_rn(myp, st.my);
    st.Sff = __fadd_rn(__fadd_rn(st.Sff, sff), __fmul_rn(__fmul_rn(ef, ef), w));
    st.Syy = __fadd_rn(__fadd_rn(st.Syy, syy), __fmul_rn(__fmul_rn(ey, ey), w));
    st.Sfy = __fadd_rn(__fadd_rn(st.Sfy, sfy), __fmul_rn(__fmul_rn(ef, ey), w));
    st.mf = __fadd_rn(st.mf, __fmul_rn(ef, __fdiv_rn(np_, nt)));
    st.my = __fadd_rn(st.my, __fmul_rn(ey, __fdiv_rn(np_, nt)));
    st.n = nt;
}

// The target's side of a full pass without invalid targets does not depend on the individual: ky, gy, the centred
// targets dy[k] and Syy, computed once per CTA by one warp with the arithmetic and order of corr_sums<true>.
struct CorrYPass { float ky, gy, syy, pad; };
__device__ __forceinline__ void corr_y_side(const float (&y)[16], float (&dy)[16], CorrYPass& yp)
{
    yp.ky = __shfl_sync(0xffffffffu, y[0], 0);
    float sy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) sy = __fadd_rn(sy, __fsub_rn(y[k], yp.ky));
    yp.gy = __fdiv_rn(warp_sum(sy), 512.f);
    float syy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) { dy[k] = __fsub_rn(__fsub_rn(y[k], yp.ky), yp.gy); syy = __fmaf_rn(dy[k], dy[k], syy); }
    yp.syy = warp_sum(syy);
    yp.pad = 0.f;
}

// A full pass without invalid targets, the target's side precomputed (dy4: this lane's float4 of block g at dy4[g * 32]).
// Returns false, having changed nothing, when an output of the pass is not finite (the sum of the shifted outputs is
// then not finite either): the caller takes corr_pass. The outputs' side is corr_sums<true> instruction for instruction.
__device__ __forceinline__ bool corr_pass_pre(const float (&f)[16], const float4* dy4, const CorrYPass& yp, CorrState& st)
{
    const float kf = __shfl_sync(0xffffffffu, f[0], 0);
    float sf = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) sf = __fadd_rn(sf, __fsub_rn(f[k], kf));
    const float tot = warp_sum(sf);
    if (!__all_sync(0xffffffffu, finite32(tot))) return false;     // the butterfly leaves the same bits in every lane; the vote tells ptxas so
    const float gf = __fdiv_rn(tot, 512.f);
    float sff = 0.f, sfy = 0.f;
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const float4 d4 = dy4[g * 32];
        const float dd[4] = { d4.x, d4.y, d4.z, d4.w };
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float df = __fsub_rn(__fsub_rn(f[4 * g + e], kf), gf);
            sff = __fmaf_rn(df, df, sff); sfy = __fmaf_rn(df, dd[e], sfy);
        }
    }
    sff = warp_sum(sff); sfy = warp_sum(sfy);
    corr_merge(st, 512.f, __fadd_rn(kf, gf), __fadd_rn(yp.ky, yp.gy), sff, yp.syy, sfy);
    return true;
}

// the two summation passes over the valid pairs of one 512-case pass; ALL: every pair is valid (no tests), the
// arithmetic and its order are those of the masked version, so both give the same bits
template <bool ALL>
__device__ __forceinline__ void corr_sums(const float (&f)[16], const float (&y)[16], uint32_t vmask, float kf, float ky, float np_,
                                          float& gf, float& gy, float& sff, float& syy, float& sfy)
{
    float sf = 0.f, sy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) if (ALL || ((vmask >> k) & 1u)) { sf = __fadd_rn(sf, __fsub_rn(f[k], kf)); sy = __fadd_rn(sy, __fsub_rn(y[k], ky)); }
    gf = __fdiv_rn(warp_sum(sf), np_); gy = __fdiv_rn(warp_sum(sy), np_);
    sff = 0.f; syy = 0.f; sfy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) if (ALL || ((vmask >> k) & 1u)) {
        const float df = __fsub_rn(__fsub_rn(f[k], kf), gf), dy = __fsub_rn(__fsub_rn(y[k], ky), gy);
        sff = __fmaf_rn(df, df, sff); syy = __fmaf_rn(dy, dy, syy); sfy = __fmaf_rn(df, dy, sfy);
    }
    sff = warp_sum(sff); syy = warp_sum(syy); sfy = warp_sum(sfy);
}

// f[k], y[k]: case c0 + (k / 4) * 128 + lane * 4 + (k % 4); cases >= n do not count.
// y_finite (warp-uniform): every target of the call is finite, so a full pass whose outputs are all finite has no
// invalid pair and takes the test-free version.
__device__ __forceinline__ void corr_pass(const float (&f)[16], const float (&y)[16], int c0, int n, int lane, bool y_finite, CorrState& st)
{
    float gf, gy, sff, syy, sfy, kf, ky, np_;
    bool all = y_finite && c0 + 512 <= n;
    if (all) {
        float z = 0.f;                                             // 0 * f is NaN exactly when f is not finite
#pragma unroll
        for (int k = 0; k < 16; ++k) z = __fmaf_rn(f[k], 0.f, z);
        all = __all_sync(0xffffffffu, z == 0.f);
    }
    if (all) {
        np_ = 512.f;
        kf = __shfl_sync(0xffffffffu, f[0], 0); ky = __shfl_sync(0xffffffffu, y[0], 0);
        corr_sums<true>(f, y, 0xffffu, kf, ky, np_, gf, gy, sff, syy, sfy);
    } else {
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
        if (!__any_sync(0xffffffffu, nvp != 0)) return;            // warp-uniform (the vote tells ptxas so)
        // shift: the first valid pair of the pass
        kf = 0.f; ky = 0.f;
#pragma unroll
        for (int k = 15; k >= 0; --k) if ((vmask >> k) & 1u) { kf = f[k]; ky = y[k]; }
        const int first = __ffs(__ballot_sync(0xffffffffu, vmask != 0)) - 1;
        kf = __shfl_sync(0xffffffffu, kf, first);
        ky = __shfl_sync(0xffffffffu, ky, first);
        np_ = (float)nvp;
        corr_sums<false>(f, y, vmask, kf, ky, np_, gf, gy, sff, syy, sfy);
    }
    corr_merge(st, np_, __fadd_rn(kf, gf), __fadd_rn(ky, gy), sff, syy, sfy);
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
