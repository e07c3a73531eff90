// ops.cuh — per-element fp32 semantics of the Beagle commands on the device (D2, §6).
//
// Table 3 of the paper gives the meanings; the protected forms are north_star's
// (R4, R5). Accuracy contract of each implementation, u = 2^-24:
//   ADD SUB MUL  IEEE round-to-nearest (never contracted into FMA: separate GP commands)
//   DIV   a * rcp.approx.ftz(b)            rel <= 3.5u; |b| > 2^126: + |a| * 2^-126 absolute
//   SQRT  sqrt.approx.ftz(|a|)             rel <= 3u; denormal |a| flushes to 0 (abs <= 1.1e-19)
//   EXP   ex2.approx.ftz(min.NaN(a,80)*log2e)   rel <= (6 + 2.5|t|)u, results < 2^-126 flush to 0
//   LOG   lg2.approx.ftz(|a|) * ln2        abs <= 4u + 5u|v|
//   SIN COS  sin/cos.approx.ftz            abs <= (12 + 3|a|)u
// The protected tests are selects, not branches, so a warp never diverges on data.
#pragma once
#include <stdint.h>
#include <string.h>

namespace beagle {

constexpr float kEps = 1e-6f; // DESIGN.md D2: protection threshold, strict '<' on |.|

__device__ __forceinline__ float mufu_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_lg2(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_sin(float x) { float r; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float mufu_cos(float x) { float r; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float min_nan(float a, float b) { float r; asm("min.NaN.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b)); return r; }

__device__ __forceinline__ float op_add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float op_sub(float a, float b) { return __fsub_rn(a, b); }            // second-top - top
__device__ __forceinline__ float op_mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float op_div(float a, float b) {                                      // PAPER.md:238, protected
    float q = __fmul_rn(a, mufu_rcp(b));
    return fabsf(b) < kEps ? 1.0f : q;   // NaN compares false -> the arithmetic branch, NaN propagates
}
__device__ __forceinline__ float op_sin(float a) { return mufu_sin(a); }
__device__ __forceinline__ float op_cos(float a) { return mufu_cos(a); }
__device__ __forceinline__ float op_log(float a) {                                               // PAPER.md:253, protected
    float v = __fmul_rn(mufu_lg2(fabsf(a)), 0.693147180559945309f);
    return fabsf(a) < kEps ? 0.0f : v;
}
__device__ __forceinline__ float op_sqrt(float a) { return mufu_sqrt(fabsf(a)); }                // PAPER.md:249, protected
__device__ __forceinline__ float op_exp(float a) {                                               // PAPER.md:275, clamped (R5)
    return mufu_ex2(__fmul_rn(min_nan(a, 80.0f), 1.44269504088896341f));
}

__device__ __forceinline__ float op_sign(float a) { return -a; }                                 // PAPER.md:243, exact
__device__ __forceinline__ float op_square(float a) { return __fmul_rn(a, a); }
__device__ __forceinline__ float op_cube(float a) { return __fmul_rn(__fmul_rn(a, a), a); }      // (a*a)*a

// unprotected, as the paper's are; the CUDA math library's accurate versions (documented 1 4 2 2 2 2 ulp)
__device__ __forceinline__ float op_cbrt(float a) { return cbrtf(a); }
__device__ __forceinline__ float op_tan(float a) { return tanf(a); }
__device__ __forceinline__ float op_arcsin(float a) { return asinf(a); }
__device__ __forceinline__ float op_arccos(float a) { return acosf(a); }
__device__ __forceinline__ float op_arctan(float a) { return atanf(a); }
__device__ __forceinline__ float op_tanh(float a) { return tanhf(a); }

__device__ __forceinline__ float op_pow(float a, float b) { return powf(a, b); }

// token fields (D1)
__host__ __device__ __forceinline__ uint32_t tok_op(uint32_t w) { return w & 0xFFu; }
__host__ __device__ __forceinline__ uint32_t tok_arg(uint32_t w) { return w >> 8; }

// What compile_general needs in both worlds: it is compiled for the host too, so that the rules of the whole language and the
// records they emit can be tested without a device (beagle_debug_compile, test only; the device code is unchanged by this).
// On the host the reciprocal of a constant divisor is the IEEE one: a stand-in for the division handler's rcp.approx, which
// only the device has (a host-compiled record of "x / c" therefore carries 1/c to half an ulp instead of the device's bits).
#ifdef __CUDA_ARCH__
#define BG_LDG(p) __ldg(p)
__device__ __forceinline__ uint32_t f32_bits(float f) { return __float_as_uint(f); }
__device__ __forceinline__ float bits_f32(uint32_t u) { return __uint_as_float(u); }
__device__ __forceinline__ float rcp_of_const(float c) { return mufu_rcp(c); }
#else
#define BG_LDG(p) (*(p))
inline uint32_t f32_bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }
inline float bits_f32(uint32_t u) { float f; memcpy(&f, &u, 4); return f; }
inline float rcp_of_const(float c) { return 1.0f / c; }
#endif

} // namespace beagle
