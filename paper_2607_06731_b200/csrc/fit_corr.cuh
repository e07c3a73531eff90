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
#include <math.h>


// Every function here is compiled for the host too (beagle_debug_corr, test only: a warp of 32 OS threads under the SIMT emulator of
// simt_host.inc). The arithmetic is IEEE single precision throughout (add, sub, mul, div, fma, all round-to-nearest), so the host build
// computes the device's bits. The device build is these intrinsics, token for token what it was; on the host the same operations written
// plainly, and the warp collectives go to the emulator through the functions declared below (defined in simt_host.inc).
#ifdef __CUDA_ARCH__
#define CF_ADD(a, b) __fadd_rn(a, b)
#define CF_SUB(a, b) __fsub_rn(a, b)
#define CF_MUL(a, b) __fmul_rn(a, b)
#define CF_DIV(a, b) __fdiv_rn(a, b)
#define CF_FMA(a, b, c) __fmaf_rn(a, b, c)
#define CF_SHFL_XOR(v, m) __shfl_xor_sync(0xffffffffu, v, m)
#define CF_SHFL(v, l) __shfl_sync(0xffffffffu, v, l)
#define CF_ALL(p) __all_sync(0xffffffffu, p)
#define CF_ANY(p) __any_sync(0xffffffffu, p)
#define CF_BALLOT(p) __ballot_sync(0xffffffffu, p)
#define CF_POPC(x) __popc(x)
#define CF_FFS(x) __ffs(x)
#define CF_INF __int_as_float(0x7f800000)
#else
#define CF_ADD(a, b) ((float)(a) + (float)(b))
#define CF_SUB(a, b) ((float)(a) - (float)(b))
#define CF_MUL(a, b) ((float)(a) * (float)(b))
#define CF_DIV(a, b) ((float)(a) / (float)(b))
#define CF_FMA(a, b, c) fmaf(a, b, c)
#define CF_SHFL_XOR(v, m) beagle::simt_warp::shfl_xor(v, m)
#define CF_SHFL(v, l) beagle::simt_warp::shfl(v, l)
#define CF_ALL(p) beagle::simt_warp::all(p)
#define CF_ANY(p) beagle::simt_warp::any(p)
#define CF_BALLOT(p) beagle::simt_warp::ballot(p)
#define CF_POPC(x) __builtin_popcount(x)
#define CF_FFS(x) __builtin_ffs((int)(x))
#define CF_INF INFINITY
#endif
namespace beagle { namespace simt_warp {       // the calling OS thread's lane of the emulated warp (simt_host.inc)
float shfl_xor(float v, int m); int shfl_xor(int v, int m); float shfl(float v, int lane); bool all(bool p); bool any(bool p); unsigned int ballot(bool p);
} }

namespace beagle {

// The running state over the passes (warp-uniform). The mean of the outputs so far is kf + gf: kf is the shift of the first pass that had
// valid pairs (one of its outputs), gf the small offset from it; the same for the targets. Kept as two numbers because a mean of
// magnitude m rounded to one float is off by up to m u, and the merge below needs the DIFFERENCE of two means to the accuracy of the
// data's spread, not of its offset (outputs like 1e6 + x: found by the host build of this file against the oracle's bound).
struct CorrState { float n, kf, ky, gf, gy, Sff, Syy, Sfy; int c1; };

__host__ __device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v = CF_ADD(v, CF_SHFL_XOR(v, m));
    return v;
}

__host__ __device__ __forceinline__ bool finite32(float v) { return fabsf(v) < CF_INF; }

// merge the centred sums of one pass (np_ valid pairs, means kfp + gfp and kyp + gyp) into the running state (Chan et al.'s pairwise
// update). The difference of the means is taken shift from shift (two data values: exact when they are within a factor of two of each
// other, and otherwise large compared with its own rounding) plus offset from offset (small numbers).
__host__ __device__ __forceinline__ void corr_merge(CorrState& st, float np_, float kfp, float gfp, float kyp, float gyp, float sff, float syy, float sfy)
{
    if (CF_ALL(st.n == 0.f)) { st.n = np_; st.kf = kfp; st.gf = gfp; st.ky = kyp; st.gy = gyp; st.Sff = sff; st.Syy = syy; st.Sfy = sfy; return; }
    const float nt = CF_ADD(st.n, np_), w = CF_DIV(CF_MUL(st.n, np_), nt);
    const float ef = CF_ADD(CF_SUB(kfp, st.kf), CF_SUB(gfp, st.gf)), ey = CF_ADD(CF_SUB(kyp, st.ky), CF_SUB(gyp, st.gy));
    st.Sff = CF_ADD(CF_ADD(st.Sff, sff), CF_MUL(CF_MUL(ef, ef), w));
    st.Syy = CF_ADD(CF_ADD(st.Syy, syy), CF_MUL(CF_MUL(ey, ey), w));
    st.Sfy = CF_ADD(CF_ADD(st.Sfy, sfy), CF_MUL(CF_MUL(ef, ey), w));
    st.gf = CF_ADD(st.gf, CF_MUL(ef, CF_DIV(np_, nt)));
    st.gy = CF_ADD(st.gy, CF_MUL(ey, CF_DIV(np_, nt)));
    st.n = nt;
}

// The target's side of a full pass without invalid targets does not depend on the individual: ky, gy, the centred
// targets dy[k] and Syy, computed once per CTA by one warp with the arithmetic and order of corr_sums<true>.
struct CorrYPass { float ky, gy, syy, pad; };
__host__ __device__ __forceinline__ void corr_y_side(const float (&y)[16], float (&dy)[16], CorrYPass& yp)
{
    yp.ky = CF_SHFL(y[0], 0);
    float sy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) sy = CF_ADD(sy, CF_SUB(y[k], yp.ky));
    yp.gy = CF_DIV(warp_sum(sy), 512.f);
    float syy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) { dy[k] = CF_SUB(CF_SUB(y[k], yp.ky), yp.gy); syy = CF_FMA(dy[k], dy[k], syy); }
    yp.syy = warp_sum(syy);
    yp.pad = 0.f;
}

// A full pass without invalid targets, the target's side precomputed (dy4: this lane's float4 of block g at dy4[g * 32]).
// Returns false, having changed nothing, when an output of the pass is not finite (the sum of the shifted outputs is
// then not finite either): the caller takes corr_pass. The outputs' side is corr_sums<true> instruction for instruction.
__host__ __device__ __forceinline__ bool corr_pass_pre(const float (&f)[16], const float4* dy4, const CorrYPass& yp, CorrState& st)
{
    const float kf = CF_SHFL(f[0], 0);
    float sf = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) sf = CF_ADD(sf, CF_SUB(f[k], kf));
    const float tot = warp_sum(sf);
    if (!CF_ALL(finite32(tot))) return false;     // the butterfly leaves the same bits in every lane; the vote tells ptxas so
    const float gf = CF_DIV(tot, 512.f);
    float sff = 0.f, sfy = 0.f;
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const float4 d4 = dy4[g * 32];
        const float dd[4] = { d4.x, d4.y, d4.z, d4.w };
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float df = CF_SUB(CF_SUB(f[4 * g + e], kf), gf);
            sff = CF_FMA(df, df, sff); sfy = CF_FMA(df, dd[e], sfy);
        }
    }
    sff = warp_sum(sff); sfy = warp_sum(sfy);
    corr_merge(st, 512.f, kf, gf, yp.ky, yp.gy, sff, yp.syy, sfy);
    return true;
}

// the two summation passes over the valid pairs of one 512-case pass; ALL: every pair is valid (no tests), the
// arithmetic and its order are those of the masked version, so both give the same bits
template <bool ALL>
__host__ __device__ __forceinline__ void corr_sums(const float (&f)[16], const float (&y)[16], uint32_t vmask, float kf, float ky, float np_,
                                          float& gf, float& gy, float& sff, float& syy, float& sfy)
{
    float sf = 0.f, sy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) if (ALL || ((vmask >> k) & 1u)) { sf = CF_ADD(sf, CF_SUB(f[k], kf)); sy = CF_ADD(sy, CF_SUB(y[k], ky)); }
    gf = CF_DIV(warp_sum(sf), np_); gy = CF_DIV(warp_sum(sy), np_);
    sff = 0.f; syy = 0.f; sfy = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) if (ALL || ((vmask >> k) & 1u)) {
        const float df = CF_SUB(CF_SUB(f[k], kf), gf), dy = CF_SUB(CF_SUB(y[k], ky), gy);
        sff = CF_FMA(df, df, sff); syy = CF_FMA(dy, dy, syy); sfy = CF_FMA(df, dy, sfy);
    }
    sff = warp_sum(sff); syy = warp_sum(syy); sfy = warp_sum(sfy);
}

// f[k], y[k]: case c0 + (k / 4) * 128 + lane * 4 + (k % 4); cases >= n do not count.
// y_finite (warp-uniform): every target of the call is finite, so a full pass whose outputs are all finite has no
// invalid pair and takes the test-free version.
__host__ __device__ __forceinline__ void corr_pass(const float (&f)[16], const float (&y)[16], int c0, int n, int lane, bool y_finite, CorrState& st)
{
    float gf, gy, sff, syy, sfy, kf, ky, np_;
    bool all = y_finite && c0 + 512 <= n;
    if (all) {
        float z = 0.f;                                             // 0 * f is NaN exactly when f is not finite
#pragma unroll
        for (int k = 0; k < 16; ++k) z = CF_FMA(f[k], 0.f, z);
        all = CF_ALL(z == 0.f);
    }
    if (all) {
        np_ = 512.f;
        kf = CF_SHFL(f[0], 0); ky = CF_SHFL(y[0], 0);
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
        int pack = CF_POPC(vmask) | (c1l << 16);
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) pack += CF_SHFL_XOR(pack, m);
        st.c1 += pack >> 16;
        const int nvp = pack & 0xffff;
        if (!CF_ANY(nvp != 0)) return;            // warp-uniform (the vote tells ptxas so)
        // shift: the first valid pair of the pass
        kf = 0.f; ky = 0.f;
#pragma unroll
        for (int k = 15; k >= 0; --k) if ((vmask >> k) & 1u) { kf = f[k]; ky = y[k]; }
        const int first = CF_FFS(CF_BALLOT(vmask != 0)) - 1;
        kf = CF_SHFL(kf, first);
        ky = CF_SHFL(ky, first);
        np_ = (float)nvp;
        corr_sums<false>(f, y, vmask, kf, ky, np_, gf, gy, sff, syy, sfy);
    }
    corr_merge(st, np_, kf, gf, ky, gy, sff, syy, sfy);
}

__host__ __device__ __forceinline__ float corr_finish(const CorrState& st, int n, int len, float M, float tax)
{
    float r2 = 0.f;
    if (st.n >= 2.f && st.Sff > 0.f && st.Syy > 0.f) r2 = CF_MUL(CF_DIV(st.Sfy, st.Sff), CF_DIV(st.Sfy, st.Syy));   // no overflow of Sff * Syy
    const int c2 = n - (int)st.n - st.c1;
    const float score = CF_SUB(CF_MUL(CF_MUL(M, CF_MUL(r2, r2)), st.n), CF_MUL(M, (float)(st.c1 - c2)));
    return CF_FMA(-tax, (float)len, score);
}

} // namespace beagle
