// interp.cuh — the hot loop (a6) as ONE inline-PTX block: a threaded-code interpreter of the micro-ops of
// uop.cuh, 16 fitness cases per lane. DESIGN.md §7.
//
// Why PTX: the loop must (1) keep acc[16] and s[D][16] in fixed registers for its whole life, (2) dispatch
// with one indexed branch per micro-op (brx.idx -> SASS BRX through one jump table), replicated at the end of
// every handler so that the next handler's address is looked up while the current one computes, and (3) stay
// small enough for the instruction cache. nvcc's optimiser does none of the three for a C++ switch of this
// size (it emits compare chains and copies the whole register state at the merge point), so the handlers are
// written out here, by preprocessor macros, and ptxas only allocates registers and schedules.
//
// Per-command arithmetic is instruction for instruction that of ops.cuh (same PTX opcodes, same constants),
// so per-case outputs are bit-identical to the C++ kernels that use ops.cuh (k_eval_blockwise).
//
// Register names inside the block: a<k> accumulator, s<S>_<k> slot S, x<k> staged variable values,
// t<k>/q<k>/p<k> temporaries, (ux,uy) current micro-op, (nx,ny) the prefetched next one, pc its address.
#pragma once
#include "uop.cuh"

// ---- repetition helpers -------------------------------------------------------------------------------
#define BGI_K16(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15)
#define BGI_K16S(M, S) M(S,0) M(S,1) M(S,2) M(S,3) M(S,4) M(S,5) M(S,6) M(S,7) M(S,8) M(S,9) M(S,10) M(S,11) M(S,12) M(S,13) M(S,14) M(S,15)

// ---- constants (hex fp32) -------------------------------------------------------------------------------
#define BGI_EPS   "0f358637BD"   /* 1e-6f                     DESIGN.md D2 */
#define BGI_ONE   "0f3F800000"
#define BGI_ZERO  "0f00000000"
#define BGI_LN2   "0f3F317218"   /* 0.693147180559945309f     ops.cuh op_log */
#define BGI_LOG2E "0f3FB8AA3B"   /* 1.44269504088896341f      ops.cuh op_exp */
#define BGI_80    "0f42A00000"

// ---- per-element command bodies: DST = f(A, B); temporaries indexed by k ---------------------------------
#define BGI_DIV(DST, A, B, k) \
    "rcp.approx.ftz.f32 t" #k ", " B ";\n" \
    "mul.rn.f32 q" #k ", " A ", t" #k ";\n" \
    "abs.f32 t" #k ", " B ";\n" \
    "setp.lt.f32 p" #k ", t" #k ", " BGI_EPS ";\n" \
    "selp.f32 " DST ", " BGI_ONE ", q" #k ", p" #k ";\n"
#define BGI_SIN(k)  "sin.approx.ftz.f32 a" #k ", a" #k ";\n"
#define BGI_COS(k)  "cos.approx.ftz.f32 a" #k ", a" #k ";\n"
#define BGI_SQRT(k) "abs.f32 t" #k ", a" #k ";\n" "sqrt.approx.ftz.f32 a" #k ", t" #k ";\n"
#define BGI_LOG(k) \
    "abs.f32 t" #k ", a" #k ";\n" \
    "lg2.approx.ftz.f32 q" #k ", t" #k ";\n" \
    "mul.rn.f32 q" #k ", q" #k ", " BGI_LN2 ";\n" \
    "setp.lt.f32 p" #k ", t" #k ", " BGI_EPS ";\n" \
    "selp.f32 a" #k ", " BGI_ZERO ", q" #k ", p" #k ";\n"
#define BGI_EXP(k) \
    "min.NaN.f32 t" #k ", a" #k ", " BGI_80 ";\n" \
    "mul.rn.f32 t" #k ", t" #k ", " BGI_LOG2E ";\n" \
    "ex2.approx.ftz.f32 a" #k ", t" #k ";\n"

// operand = staged variable (x<k>)
#define BGI_LOADX(k) "mov.f32 a" #k ", x" #k ";\n"
#define BGI_ADDX(k)  "add.rn.f32 a" #k ", a" #k ", x" #k ";\n"
#define BGI_SUBX(k)  "sub.rn.f32 a" #k ", a" #k ", x" #k ";\n"
#define BGI_MULX(k)  "mul.rn.f32 a" #k ", a" #k ", x" #k ";\n"
#define BGI_XSUB(k)  "sub.rn.f32 a" #k ", x" #k ", a" #k ";\n"
#define BGI_DIVX(k)  BGI_DIV("a" #k, "a" #k, "x" #k, k)
#define BGI_XDIV(k)  BGI_DIV("a" #k, "x" #k, "a" #k, k)
// operand = constant (cv)
#define BGI_CONST(k) "mov.f32 a" #k ", cv;\n"
#define BGI_ADDC(k)  "add.rn.f32 a" #k ", a" #k ", cv;\n"
#define BGI_SUBC(k)  "sub.rn.f32 a" #k ", a" #k ", cv;\n"
#define BGI_MULC(k)  "mul.rn.f32 a" #k ", a" #k ", cv;\n"
#define BGI_CSUB(k)  "sub.rn.f32 a" #k ", cv, a" #k ";\n"
#define BGI_DIVC(k)  BGI_DIV("a" #k, "a" #k, "cv", k)
#define BGI_CDIV(k)  BGI_DIV("a" #k, "cv", "a" #k, k)
// operand = slot S
#define BGI_PUSH(S, k)  "mov.f32 s" #S "_" #k ", a" #k ";\n"
#define BGI_ADDS(S, k)  "add.rn.f32 a" #k ", s" #S "_" #k ", a" #k ";\n"
#define BGI_SUBS(S, k)  "sub.rn.f32 a" #k ", s" #S "_" #k ", a" #k ";\n"
#define BGI_MULS(S, k)  "mul.rn.f32 a" #k ", s" #S "_" #k ", a" #k ";\n"
#define BGI_RSUBS(S, k) "sub.rn.f32 a" #k ", a" #k ", s" #S "_" #k ";\n"
#define BGI_DIVS(S, k)  BGI_DIV("a" #k, "s" #S "_" #k, "a" #k, k)
#define BGI_RDIVS(S, k) BGI_DIV("a" #k, "a" #k, "s" #S "_" #k, k)

// ---- handler frame ---------------------------------------------------------------------------------------
// entry: (ux,uy) = this micro-op, pc = its shared-memory address. The next micro-op is requested first; the
// dispatch at the end looks its handler up and branches.
#define BGI_ENTER(L) "L_" #L "_%=:\n" "ld.shared.v2.b32 {nx, ny}, [pc+8];\n"
#define BGI_LEAVE \
    "add.u32 pc, pc, 8;\n" \
    "and.b32 h, nx, 255;\n" \
    "mov.b32 ux, nx;\n" \
    "mov.b32 uy, ny;\n" \
    "brx.idx h, TBL_%=;\n"
#define BGI_GETX \
    "shr.u32 o, ux, 8;\n" \
    "add.u32 o, o, xp;\n" \
    "ld.shared.v4.f32 {x0, x1, x2, x3}, [o];\n" \
    "ld.shared.v4.f32 {x4, x5, x6, x7}, [o+512];\n" \
    "ld.shared.v4.f32 {x8, x9, x10, x11}, [o+1024];\n" \
    "ld.shared.v4.f32 {x12, x13, x14, x15}, [o+1536];\n"
#define BGI_GETC "mov.b32 cv, uy;\n"

#define BGI_H_PLAIN(L, BODY) BGI_ENTER(L) BGI_K16(BODY) BGI_LEAVE
#define BGI_H_X(L, BODY)     BGI_ENTER(L) BGI_GETX BGI_K16(BODY) BGI_LEAVE
#define BGI_H_C(L, BODY)     BGI_ENTER(L) BGI_GETC BGI_K16(BODY) BGI_LEAVE

#define BGI_FIXED_HANDLERS \
    BGI_H_X(LOADX, BGI_LOADX) BGI_H_C(CONST, BGI_CONST) \
    BGI_H_PLAIN(SIN, BGI_SIN) BGI_H_PLAIN(COS, BGI_COS) BGI_H_PLAIN(LOG, BGI_LOG) \
    BGI_H_PLAIN(SQRT, BGI_SQRT) BGI_H_PLAIN(EXP, BGI_EXP) \
    BGI_H_X(ADDX, BGI_ADDX) BGI_H_X(SUBX, BGI_SUBX) BGI_H_X(MULX, BGI_MULX) BGI_H_X(DIVX, BGI_DIVX) \
    BGI_H_X(XSUB, BGI_XSUB) BGI_H_X(XDIV, BGI_XDIV) \
    BGI_H_C(ADDC, BGI_ADDC) BGI_H_C(SUBC, BGI_SUBC) BGI_H_C(MULC, BGI_MULC) BGI_H_C(DIVC, BGI_DIVC) \
    BGI_H_C(CSUB, BGI_CSUB) BGI_H_C(CDIV, BGI_CDIV)

#define BGI_SLOT_HANDLERS(S) \
    BGI_ENTER(PUSHX##S) BGI_GETX BGI_K16S(BGI_PUSH, S) BGI_K16(BGI_LOADX) BGI_LEAVE \
    BGI_ENTER(PUSHC##S) BGI_GETC BGI_K16S(BGI_PUSH, S) BGI_K16(BGI_CONST) BGI_LEAVE \
    BGI_ENTER(ADDS##S) BGI_K16S(BGI_ADDS, S) BGI_LEAVE \
    BGI_ENTER(SUBS##S) BGI_K16S(BGI_SUBS, S) BGI_LEAVE \
    BGI_ENTER(MULS##S) BGI_K16S(BGI_MULS, S) BGI_LEAVE \
    BGI_ENTER(DIVS##S) BGI_K16S(BGI_DIVS, S) BGI_LEAVE \
    BGI_ENTER(RSUBS##S) BGI_K16S(BGI_RSUBS, S) BGI_LEAVE \
    BGI_ENTER(RDIVS##S) BGI_K16S(BGI_RDIVS, S) BGI_LEAVE

#define BGI_SLOT_DECL(S) ".reg .f32 s" #S "_<16>;\n"

// jump table rows: 8 entries per slot-indexed family; slots the instantiation does not have go to END
#define BGI_T(L) "L_" #L "_%=, "
#define BGI_FAMILY5(F) BGI_T(F##0) BGI_T(F##1) BGI_T(F##2) BGI_T(F##3) BGI_T(F##4) BGI_T(END) BGI_T(END) BGI_T(END)
#define BGI_FAMILY8(F) BGI_T(F##0) BGI_T(F##1) BGI_T(F##2) BGI_T(F##3) BGI_T(F##4) BGI_T(F##5) BGI_T(F##6) BGI_T(F##7)
#define BGI_TABLE(FAMILY) \
    "TBL_%=: .branchtargets " \
    BGI_T(END) BGI_T(LOADX) BGI_T(CONST) BGI_T(SIN) BGI_T(COS) BGI_T(LOG) BGI_T(SQRT) BGI_T(EXP) \
    BGI_T(ADDX) BGI_T(SUBX) BGI_T(MULX) BGI_T(DIVX) BGI_T(XSUB) BGI_T(XDIV) \
    BGI_T(ADDC) BGI_T(SUBC) BGI_T(MULC) BGI_T(DIVC) BGI_T(CSUB) BGI_T(CDIV) \
    FAMILY(PUSHX) FAMILY(PUSHC) FAMILY(ADDS) FAMILY(SUBS) FAMILY(MULS) FAMILY(DIVS) FAMILY(RSUBS) FAMILY(RDIVS) \
    "L_END_%=;\n"

#define BGI_OUT(k) "mov.f32 %" #k ", a" #k ";\n"

// The whole block. SLOT_DECLS / SLOT_CODE: BGI_SLOT_DECL / BGI_SLOT_HANDLERS over the instantiation's slots.
// Operands: %0..%15 = acc out, %16 = shared address of the micro-ops, %17 = shared address of this lane's cases.
#define BGI_ASM(SLOT_DECLS, SLOT_CODE, FAMILY) \
    "{\n" \
    ".reg .f32 a<16>, x<16>, t<16>, q<16>, cv;\n" \
    ".reg .pred p<16>;\n" \
    ".reg .b32 ux, uy, nx, ny, pc, h, o, xp;\n" \
    SLOT_DECLS \
    BGI_TABLE(FAMILY) \
    "mov.u32 pc, %16;\n" \
    "mov.u32 xp, %17;\n" \
    "ld.shared.v2.b32 {ux, uy}, [pc];\n" \
    "and.b32 h, ux, 255;\n" \
    "brx.idx h, TBL_%=;\n" \
    BGI_FIXED_HANDLERS \
    SLOT_CODE \
    "L_END_%=:\n" \
    BGI_K16(BGI_OUT) \
    "}\n"

#define BGI_ACC_OUT(A) "=f"(A[0]), "=f"(A[1]), "=f"(A[2]), "=f"(A[3]), "=f"(A[4]), "=f"(A[5]), "=f"(A[6]), "=f"(A[7]), \
                       "=f"(A[8]), "=f"(A[9]), "=f"(A[10]), "=f"(A[11]), "=f"(A[12]), "=f"(A[13]), "=f"(A[14]), "=f"(A[15])

namespace beagle {

// acc[k] = the program's output on case (c0 + (k/4)*128 + lane*4 + k%4)
__device__ __forceinline__ void interp_run_d5(uint32_t ubuf, uint32_t xp, float (&acc)[16])
{
    asm volatile(BGI_ASM(BGI_SLOT_DECL(0) BGI_SLOT_DECL(1) BGI_SLOT_DECL(2) BGI_SLOT_DECL(3) BGI_SLOT_DECL(4),
                         BGI_SLOT_HANDLERS(0) BGI_SLOT_HANDLERS(1) BGI_SLOT_HANDLERS(2) BGI_SLOT_HANDLERS(3) BGI_SLOT_HANDLERS(4),
                         BGI_FAMILY5)
                 : BGI_ACC_OUT(acc) : "r"(ubuf), "r"(xp) : "memory");
}

__device__ __forceinline__ void interp_run_d8(uint32_t ubuf, uint32_t xp, float (&acc)[16])
{
    asm volatile(BGI_ASM(BGI_SLOT_DECL(0) BGI_SLOT_DECL(1) BGI_SLOT_DECL(2) BGI_SLOT_DECL(3) BGI_SLOT_DECL(4)
                         BGI_SLOT_DECL(5) BGI_SLOT_DECL(6) BGI_SLOT_DECL(7),
                         BGI_SLOT_HANDLERS(0) BGI_SLOT_HANDLERS(1) BGI_SLOT_HANDLERS(2) BGI_SLOT_HANDLERS(3) BGI_SLOT_HANDLERS(4)
                         BGI_SLOT_HANDLERS(5) BGI_SLOT_HANDLERS(6) BGI_SLOT_HANDLERS(7),
                         BGI_FAMILY8)
                 : BGI_ACC_OUT(acc) : "r"(ubuf), "r"(xp) : "memory");
}

} // namespace beagle
