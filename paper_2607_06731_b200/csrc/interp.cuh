// interp.cuh — the hot loop (a6) as ONE inline-PTX block: a threaded-code interpreter of the micro-ops of
// uop.cuh, 16 fitness cases per lane. DESIGN.md §7.
//
// Why PTX: the loop must (1) keep acc[16] and s[4][16] in fixed registers for its whole life, (2) dispatch
// with one indexed branch per micro-op (brx.idx -> SASS LDC + BRX through one jump table), replicated at the
// end of every handler, with the index already in a register when the handler starts, so that the table
// lookup overlaps the handler's arithmetic, and (3) stay inside the 32 KB instruction cache level. nvcc's
// optimiser does none of the three for a C++ switch of this size (it emits compare chains and copies the
// whole register state at the merge point), so the handlers are written out here, by preprocessor macros,
// and ptxas only allocates registers and schedules.
//
// Per-command arithmetic is instruction for instruction that of ops.cuh (same PTX opcodes, same constants),
// so per-case outputs are bit-identical to the C++ kernel that uses ops.cuh (k_eval_blockwise).
//
// Register names inside the block: a<k> accumulator, s<S>_<k> slot S, x<k> staged variable values / second
// operand, t<k>/q<k>/p<k> temporaries; (h, o) = the record of the running micro-op = {handler of the NEXT
// micro-op | extra << 8, operand}; (h2, o2) the record being prefetched; pc = shared address of (h, o).
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

// ---- per-element command bodies; temporaries indexed by k ------------------------------------------------
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

// second operand in x<k> (a staged variable, or a slot copied/loaded into x)
#define BGI_LOADX(k) "mov.f32 a" #k ", x" #k ";\n"
#define BGI_ADDX(k)  "add.rn.f32 a" #k ", a" #k ", x" #k ";\n"
#define BGI_SUBX(k)  "sub.rn.f32 a" #k ", a" #k ", x" #k ";\n"
#define BGI_MULX(k)  "mul.rn.f32 a" #k ", a" #k ", x" #k ";\n"
#define BGI_XSUB(k)  "sub.rn.f32 a" #k ", x" #k ", a" #k ";\n"
#define BGI_DIVX(k)  BGI_DIV("a" #k, "a" #k, "x" #k, k)
#define BGI_XDIV(k)  BGI_DIV("a" #k, "x" #k, "a" #k, k)
// second operand = constant (cv)
#define BGI_CONST(k) "mov.f32 a" #k ", cv;\n"
#define BGI_ADDC(k)  "add.rn.f32 a" #k ", a" #k ", cv;\n"
#define BGI_SUBC(k)  "sub.rn.f32 a" #k ", a" #k ", cv;\n"
#define BGI_MULC(k)  "mul.rn.f32 a" #k ", a" #k ", cv;\n"
#define BGI_CSUB(k)  "sub.rn.f32 a" #k ", cv, a" #k ";\n"
#define BGI_DIVC(k)  BGI_DIV("a" #k, "a" #k, "cv", k)
#define BGI_CDIV(k)  BGI_DIV("a" #k, "cv", "a" #k, k)
// first operand = register slot S
#define BGI_PUSH(S, k)  "mov.f32 s" #S "_" #k ", a" #k ";\n"
#define BGI_ADDS(S, k)  "add.rn.f32 a" #k ", s" #S "_" #k ", a" #k ";\n"
#define BGI_SUBS(S, k)  "sub.rn.f32 a" #k ", s" #S "_" #k ", a" #k ";\n"
#define BGI_MULS(S, k)  "mul.rn.f32 a" #k ", s" #S "_" #k ", a" #k ";\n"
#define BGI_S2X(S, k)   "mov.f32 x" #k ", s" #S "_" #k ";\n"

// ---- handler frame ---------------------------------------------------------------------------------------
// entry: (h, o) = this micro-op's record, pc = its shared-memory address. The next record is requested
// first; the dispatch at the end branches through the table on the handler number that arrived with (h, o).
#define BGI_ENTER(L) "L_" #L "_%=:\n" "ld.shared.v2.b32 {h2, o2}, [pc+8];\n" "and.b32 hn, h, 255;\n"
#define BGI_LEAVE \
    "add.u32 pc, pc, 8;\n" \
    "mov.b32 h, h2;\n" \
    "mov.b32 o, o2;\n" \
    "brx.idx hn, TBL_%=;\n"
#define BGI_GETX \
    "add.u32 xa, o, xp;\n" \
    "ld.shared.v4.f32 {x0, x1, x2, x3}, [xa];\n" \
    "ld.shared.v4.f32 {x4, x5, x6, x7}, [xa+512];\n" \
    "ld.shared.v4.f32 {x8, x9, x10, x11}, [xa+1024];\n" \
    "ld.shared.v4.f32 {x12, x13, x14, x15}, [xa+1536];\n"
#define BGI_GETC "mov.b32 cv, o;\n"
// local slot memory: 16 floats per slot per lane at byte offset extra = h >> 8
#define BGI_MEMADDR \
    "shr.u32 e, h, 8;\n" \
    "cvt.u64.u32 ma, e;\n" \
    "add.u64 ma, ma, mbase;\n"
#define BGI_GETM BGI_MEMADDR \
    "ld.local.v4.f32 {x0, x1, x2, x3}, [ma];\n" \
    "ld.local.v4.f32 {x4, x5, x6, x7}, [ma+16];\n" \
    "ld.local.v4.f32 {x8, x9, x10, x11}, [ma+32];\n" \
    "ld.local.v4.f32 {x12, x13, x14, x15}, [ma+48];\n"
#define BGI_PUTM BGI_MEMADDR \
    "st.local.v4.f32 [ma], {a0, a1, a2, a3};\n" \
    "st.local.v4.f32 [ma+16], {a4, a5, a6, a7};\n" \
    "st.local.v4.f32 [ma+32], {a8, a9, a10, a11};\n" \
    "st.local.v4.f32 [ma+48], {a12, a13, a14, a15};\n"

#define BGI_H_PLAIN(L, BODY) BGI_ENTER(L) BGI_K16(BODY) BGI_LEAVE
#define BGI_H_X(L, BODY)     BGI_ENTER(L) BGI_GETX "B_" #L "_%=:\n" BGI_K16(BODY) BGI_LEAVE
#define BGI_H_C(L, BODY)     BGI_ENTER(L) BGI_GETC BGI_K16(BODY) BGI_LEAVE
#define BGI_GOTO(L)          "bra.uni B_" #L "_%=;\n"

#define BGI_FIXED_HANDLERS \
    BGI_H_X(LOADX, BGI_LOADX) BGI_H_C(CONST, BGI_CONST) \
    BGI_H_PLAIN(SIN, BGI_SIN) BGI_H_PLAIN(COS, BGI_COS) BGI_H_PLAIN(LOG, BGI_LOG) \
    BGI_H_PLAIN(SQRT, BGI_SQRT) BGI_H_PLAIN(EXP, BGI_EXP) \
    BGI_H_X(ADDX, BGI_ADDX) BGI_H_X(SUBX, BGI_SUBX) BGI_H_X(MULX, BGI_MULX) BGI_H_X(DIVX, BGI_DIVX) \
    BGI_H_X(XSUB, BGI_XSUB) BGI_H_X(XDIV, BGI_XDIV) \
    BGI_H_C(ADDC, BGI_ADDC) BGI_H_C(SUBC, BGI_SUBC) BGI_H_C(MULC, BGI_MULC) BGI_H_C(DIVC, BGI_DIVC) \
    BGI_H_C(CSUB, BGI_CSUB) BGI_H_C(CDIV, BGI_CDIV)

// register slot S. DIVS copies the slot into x and shares XDIV's body (acc = x / acc): the protected
// division is the longest body, and sharing it keeps the loop inside the instruction cache.
#define BGI_SLOT_HANDLERS(S) \
    BGI_ENTER(PUSHX##S) BGI_GETX BGI_K16S(BGI_PUSH, S) BGI_K16(BGI_LOADX) BGI_LEAVE \
    BGI_ENTER(PUSHC##S) BGI_GETC BGI_K16S(BGI_PUSH, S) BGI_K16(BGI_CONST) BGI_LEAVE \
    BGI_ENTER(ADDS##S) BGI_K16S(BGI_ADDS, S) BGI_LEAVE \
    BGI_ENTER(SUBS##S) BGI_K16S(BGI_SUBS, S) BGI_LEAVE \
    BGI_ENTER(MULS##S) BGI_K16S(BGI_MULS, S) BGI_LEAVE \
    BGI_ENTER(DIVS##S) BGI_K16S(BGI_S2X, S) BGI_GOTO(XDIV)

// memory slots: acc = mem op acc is "x = mem" followed by the body of acc = x op acc
#define BGI_MEM_HANDLERS \
    BGI_ENTER(PUSHXM) BGI_PUTM BGI_GETX BGI_K16(BGI_LOADX) BGI_LEAVE \
    BGI_ENTER(PUSHCM) BGI_PUTM BGI_GETC BGI_K16(BGI_CONST) BGI_LEAVE \
    BGI_ENTER(ADDM) BGI_GETM BGI_GOTO(ADDX) \
    BGI_ENTER(SUBM) BGI_GETM BGI_GOTO(XSUB) \
    BGI_ENTER(MULM) BGI_GETM BGI_GOTO(MULX) \
    BGI_ENTER(DIVM) BGI_GETM BGI_GOTO(XDIV)

#define BGI_SLOT_DECL(S) ".reg .f32 s" #S "_<16>;\n"

#define BGI_T(L) "L_" #L "_%=, "
#define BGI_FAMILY(F) BGI_T(F##0) BGI_T(F##1) BGI_T(F##2) BGI_T(F##3)
#define BGI_TABLE \
    "TBL_%=: .branchtargets " \
    BGI_T(END) BGI_T(LOADX) BGI_T(CONST) BGI_T(SIN) BGI_T(COS) BGI_T(LOG) BGI_T(SQRT) BGI_T(EXP) \
    BGI_T(ADDX) BGI_T(SUBX) BGI_T(MULX) BGI_T(DIVX) BGI_T(XSUB) BGI_T(XDIV) \
    BGI_T(ADDC) BGI_T(SUBC) BGI_T(MULC) BGI_T(DIVC) BGI_T(CSUB) BGI_T(CDIV) \
    BGI_FAMILY(PUSHX) BGI_FAMILY(PUSHC) BGI_FAMILY(ADDS) BGI_FAMILY(SUBS) BGI_FAMILY(MULS) BGI_FAMILY(DIVS) \
    BGI_T(PUSHXM) BGI_T(PUSHCM) BGI_T(ADDM) BGI_T(SUBM) BGI_T(MULM) BGI_T(DIVM) \
    "L_END_%=;\n"

#define BGI_OUT(k) "mov.f32 %" #k ", a" #k ";\n"

// Operands: %0..%15 = acc out, %16 = shared address of the records, %17 = shared address of this lane's cases.
#define BGI_ASM \
    "{\n" \
    ".reg .f32 a<16>, x<16>, t<16>, q<16>, cv;\n" \
    ".reg .pred p<16>;\n" \
    ".reg .b32 h, o, h2, o2, hn, pc, xa, xp, e;\n" \
    ".reg .b64 ma, mbase;\n" \
    ".local .align 16 .b8 slotmem[1728];\n"      /* kMemSlots * 64 */ \
    BGI_SLOT_DECL(0) BGI_SLOT_DECL(1) BGI_SLOT_DECL(2) BGI_SLOT_DECL(3) \
    BGI_TABLE \
    "mov.u32 pc, %16;\n" \
    "mov.u32 xp, %17;\n" \
    "mov.u64 mbase, slotmem;\n" \
    "ld.shared.v2.b32 {hn, o}, [pc];\n"          /* rec[0] = {handler_0, 0} */ \
    "ld.shared.v2.b32 {h, o}, [pc+8];\n"         /* rec[1] = record of micro-op 0 */ \
    "add.u32 pc, pc, 8;\n" \
    "and.b32 hn, hn, 255;\n" \
    "brx.idx hn, TBL_%=;\n" \
    BGI_FIXED_HANDLERS \
    BGI_SLOT_HANDLERS(0) BGI_SLOT_HANDLERS(1) BGI_SLOT_HANDLERS(2) BGI_SLOT_HANDLERS(3) \
    BGI_MEM_HANDLERS \
    "L_END_%=:\n" \
    BGI_K16(BGI_OUT) \
    "}\n"

#define BGI_ACC_OUT(A) "=f"(A[0]), "=f"(A[1]), "=f"(A[2]), "=f"(A[3]), "=f"(A[4]), "=f"(A[5]), "=f"(A[6]), "=f"(A[7]), \
                       "=f"(A[8]), "=f"(A[9]), "=f"(A[10]), "=f"(A[11]), "=f"(A[12]), "=f"(A[13]), "=f"(A[14]), "=f"(A[15])

namespace beagle {

static_assert(kRegSlots == 4 && kMemSlots * 64 == 1728, "interp.cuh is written for 4 register slots and 27 memory slots");

// acc[k] = the program's output on case (c0 + (k/4)*128 + lane*4 + k%4)
__device__ __forceinline__ void interp_run(uint32_t rec, uint32_t xp, float (&acc)[16])
{
    asm volatile(BGI_ASM : BGI_ACC_OUT(acc) : "r"(rec), "r"(xp) : "memory");
}

} // namespace beagle
