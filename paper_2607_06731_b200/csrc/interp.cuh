// interp.cuh — the hot loop (a6) as ONE inline-PTX block: a threaded-code interpreter of the micro-ops of
// uop.cuh, 16 fitness cases per lane. DESIGN.md §7.
//
// Why PTX: the loop must (1) keep acc[16] and the operand registers x[16] in fixed registers for its whole
// life, (2) dispatch with ONE indexed branch (brx.idx -> SASS LDC + BRX through one jump table that stays
// resident in the indexed-constant cache; a per-handler copy of the dispatch thrashes that cache: measured
// 48 % hit rate, profiles/), and (3) stay far inside the 32 KB instruction cache level. nvcc's optimiser
// does none of the three for a C++ switch of this size, so the handlers are written out here, by
// preprocessor macros, and ptxas only allocates registers and schedules.
//
// Operands come from TENSOR MEMORY: one tcgen05.ld (.32x32b.x16: this lane's 16 consecutive columns)
// delivers a variable's 16 cases, or a pushed slot, straight into x[16] (or into acc[16] for a fresh
// value). Measured on B200 (profiles/): 226 B/clk/SM against 85 B/clk/SM for the same operand fetched
// with 4 x LDS.128, one issue slot instead of five, and no shared-memory traffic at all.
// "push acc" is one tcgen05.st in front of the handler of a fresh value (the P_ entry of that handler); the
// tensor-memory slots of a warp are a stack, so the interpreter keeps their top (spt) and a pop is one
// tcgen05.ld at spt - 16.
//
// Per-command arithmetic is instruction for instruction that of ops.cuh (same PTX opcodes, same constants),
// so per-case outputs are bit-identical to the C++ kernel that uses ops.cuh (k_eval_blockwise).
//
// Register names inside the block: %0..%15 (the asm's output operands) are the accumulator, x<k> second operand, t<k>/q<k>/p<k> temporaries;
// (h, o) = the record of the micro-op being dispatched / run (uop.cuh); pc = its shared-memory address;
// xb = tensor-memory address of this pass's variable block, rb = of its reciprocal rows, sb = of this warp's
// slot block.
#pragma once
#include "uop.cuh"

// ---- repetition helpers -------------------------------------------------------------------------------
#define BGI_K16(M) M(0) M(1) M(2) M(3) M(4) M(5) M(6) M(7) M(8) M(9) M(10) M(11) M(12) M(13) M(14) M(15)
#define BGI_R16(R) R "0, " R "1, " R "2, " R "3, " R "4, " R "5, " R "6, " R "7, " R "8, " R "9, " R "10, " R "11, " R "12, " R "13, " R "14, " R "15"

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
#define BGI_SIN(k)  "sin.approx.ftz.f32 " BGI_A #k ", " BGI_A #k ";\n"
#define BGI_COS(k)  "cos.approx.ftz.f32 " BGI_A #k ", " BGI_A #k ";\n"
#define BGI_SQRT(k) "abs.f32 t" #k ", " BGI_A #k ";\n" "sqrt.approx.ftz.f32 " BGI_A #k ", t" #k ";\n"
#define BGI_LOG(k) \
    "abs.f32 t" #k ", " BGI_A #k ";\n" \
    "lg2.approx.ftz.f32 q" #k ", t" #k ";\n" \
    "mul.rn.f32 q" #k ", q" #k ", " BGI_LN2 ";\n" \
    "setp.lt.f32 p" #k ", t" #k ", " BGI_EPS ";\n" \
    "selp.f32 " BGI_A #k ", " BGI_ZERO ", q" #k ", p" #k ";\n"
#define BGI_EXP(k) \
    "min.NaN.f32 t" #k ", " BGI_A #k ", " BGI_80 ";\n" \
    "mul.rn.f32 t" #k ", t" #k ", " BGI_LOG2E ";\n" \
    "ex2.approx.ftz.f32 " BGI_A #k ", t" #k ";\n"

#define BGI_NEG(k)  "neg.f32 " BGI_A #k ", " BGI_A #k ";\n"
#define BGI_SQRE(k) "mul.rn.f32 " BGI_A #k ", " BGI_A #k ", " BGI_A #k ";\n"
#define BGI_CUBE(k) "mul.rn.f32 t" #k ", " BGI_A #k ", " BGI_A #k ";\n" "mul.rn.f32 " BGI_A #k ", t" #k ", " BGI_A #k ";\n"
#define BGI_MOVX(k) "mov.f32 " BGI_A #k ", x" #k ";\n"

// second operand in x<k> (a variable or a slot, loaded from tensor / local memory)
#define BGI_ADDX(k)  "add.rn.f32 " BGI_A #k ", " BGI_A #k ", x" #k ";\n"
#define BGI_SUBX(k)  "sub.rn.f32 " BGI_A #k ", " BGI_A #k ", x" #k ";\n"
#define BGI_MULX(k)  "mul.rn.f32 " BGI_A #k ", " BGI_A #k ", x" #k ";\n"
#define BGI_RSUBX(k) "sub.rn.f32 " BGI_A #k ", x" #k ", " BGI_A #k ";\n"
#define BGI_DIVX(k)  BGI_DIV(BGI_A #k, BGI_A #k, "x" #k, k)
#define BGI_RDIVX(k) BGI_DIV(BGI_A #k, "x" #k, BGI_A #k, k)
// second operand = constant (cv)
#define BGI_LC(k)    "mov.f32 " BGI_A #k ", cv;\n"
#define BGI_ADDC(k)  "add.rn.f32 " BGI_A #k ", " BGI_A #k ", cv;\n"
#define BGI_SUBC(k)  "sub.rn.f32 " BGI_A #k ", " BGI_A #k ", cv;\n"
#define BGI_MULC(k)  "mul.rn.f32 " BGI_A #k ", " BGI_A #k ", cv;\n"
#define BGI_RSUBC(k) "sub.rn.f32 " BGI_A #k ", cv, " BGI_A #k ";\n"
#define BGI_RDIVC(k) BGI_DIV(BGI_A #k, "cv", BGI_A #k, k)

// ---- handler frame ---------------------------------------------------------------------------------------
// entry: (h, o) = this micro-op's record, pc = its shared-memory address. NEXT replaces (h, o) by the next
// record as soon as this handler has taken what it needs from them; every handler ends at the one dispatcher.
#define BGI_NEXT    "ld.shared.v2.b32 {h, o}, [pc+8];\n" "add.u32 pc, pc, 8;\n"
#define BGI_WAITLD  "tcgen05.wait::ld.sync.aligned;\n"
#define BGI_LDTM(R, ADDR) "tcgen05.ld.sync.aligned.32x32b.x16.b32 {" BGI_R16(R) "}, [" ADDR "];\n"
#define BGI_DISPATCH "bra.uni DISP_%=;\n"
// fresh value: acc = X[colA], colA = h[31:21]
#define BGI_LXA     "shr.u32 e, h, 21;\n" "add.u32 e, e, xb;\n" BGI_LDTM(BGI_A, "e")
// x = local slot memory, 16 floats per slot per lane at byte offset o
#define BGI_GETM \
    "cvt.u64.u32 ma, o;\n" \
    "add.u64 ma, ma, mbase;\n" \
    "ld.local.v4.f32 {x0, x1, x2, x3}, [ma];\n" \
    "ld.local.v4.f32 {x4, x5, x6, x7}, [ma+16];\n" \
    "ld.local.v4.f32 {x8, x9, x10, x11}, [ma+32];\n" \
    "ld.local.v4.f32 {x12, x13, x14, x15}, [ma+48];\n"

// "push acc" in front of a fresh value: P_<entry> pushes to the warp's tensor-memory slot stack (spt), M_<entry>
// to the local-memory slot at byte offset h[20:10]; both fall / branch into the entry itself.
#define BGI_PUSHT \
    "tcgen05.st.sync.aligned.32x32b.x16.b32 [spt], {" BGI_R16(BGI_A) "};\n" \
    "tcgen05.wait::st.sync.aligned;\n" \
    "add.u32 spt, spt, 16;\n"
#define BGI_PUSHM \
    "bfe.u32 e, h, 10, 11;\n" \
    "cvt.u64.u32 ma, e;\n" \
    "add.u64 ma, ma, mbase;\n" \
    "st.local.v4.f32 [ma], {" BGI_A "0, " BGI_A "1, " BGI_A "2, " BGI_A "3};\n" \
    "st.local.v4.f32 [ma+16], {" BGI_A "4, " BGI_A "5, " BGI_A "6, " BGI_A "7};\n" \
    "st.local.v4.f32 [ma+32], {" BGI_A "8, " BGI_A "9, " BGI_A "10, " BGI_A "11};\n" \
    "st.local.v4.f32 [ma+48], {" BGI_A "12, " BGI_A "13, " BGI_A "14, " BGI_A "15};\n"
#define BGI_PUSHES(ENTRY) \
    "M_" #ENTRY "_%=:\n" BGI_PUSHM "bra.uni L_" #ENTRY "_%=;\n" \
    "P_" #ENTRY "_%=:\n" BGI_PUSHT

// acc = acc OP x: entry points for a variable (X), a tensor-memory slot (S), a local-memory slot (M) and a
// fresh first operand (LX_) share one body. J_: x is being addressed by xa; K_: x is already on its way.
#define BGI_BIN_X(OP, BODY) \
    "L_" #OP "X_%=:\n" "add.u32 xa, o, xb;\n" \
    "J_" #OP "_%=:\n" BGI_LDTM("x", "xa") \
    "K_" #OP "_%=:\n" BGI_NEXT BGI_WAITLD BGI_K16(BODY) BGI_DISPATCH
#define BGI_ENTRY_S(OP)  "L_" #OP "S_%=:\n" "sub.u32 spt, spt, 16;\n" "mov.u32 xa, spt;\n" "bra.uni J_" #OP "_%=;\n"
#define BGI_ENTRY_M(OP)  "L_" #OP "M_%=:\n" BGI_GETM "bra.uni K_" #OP "_%=;\n"
// acc = acc * (1/X)[o]: the reciprocal rows have their own base (rb); the body is MUL's
#define BGI_ENTRY_R      "L_MULR_%=:\n" "add.u32 xa, o, rb;\n" "bra.uni J_MUL_%=;\n" \
    BGI_PUSHES(LX_MULR) "L_LX_MULR_%=:\n" BGI_LXA "add.u32 xa, o, rb;\n" "bra.uni J_MUL_%=;\n"
#define BGI_ENTRY_LXX(OP) BGI_PUSHES(LX_##OP##X) "L_LX_" #OP "X_%=:\n" BGI_LXA "add.u32 xa, o, xb;\n" "bra.uni J_" #OP "_%=;\n"
// acc = acc OP c, acc = f(acc); LX_ entry: acc = X[colA] first
#define BGI_BIN_C(OP, BODY) "L_" #OP "C_%=:\n" "mov.b32 cv, o;\n" BGI_NEXT BGI_K16(BODY) BGI_DISPATCH
#define BGI_UNARY(OP, BODY) "L_" #OP "_%=:\n" BGI_NEXT BGI_K16(BODY) BGI_DISPATCH
#define BGI_ENTRY_LX(OP)  BGI_PUSHES(LX_##OP) "L_LX_" #OP "_%=:\n" BGI_LXA BGI_WAITLD "bra.uni L_" #OP "_%=;\n"

// GCL's stack commands on computed values (uop.cuh): POP (DEL) and SWAP of the slot on top, tensor or local memory
#define BGI_STM(ADDR, R) \
    "st.local.v4.f32 [" ADDR "], {" R "0, " R "1, " R "2, " R "3};\n" \
    "st.local.v4.f32 [" ADDR "+16], {" R "4, " R "5, " R "6, " R "7};\n" \
    "st.local.v4.f32 [" ADDR "+32], {" R "8, " R "9, " R "10, " R "11};\n" \
    "st.local.v4.f32 [" ADDR "+48], {" R "12, " R "13, " R "14, " R "15};\n"
#define BGI_STACKOPS \
    "L_POPS_%=:\n" "sub.u32 spt, spt, 16;\n" BGI_LDTM(BGI_A, "spt") BGI_NEXT BGI_WAITLD BGI_DISPATCH \
    "L_POPM_%=:\n" BGI_GETM BGI_NEXT BGI_K16(BGI_MOVX) BGI_DISPATCH \
    "L_SWAPS_%=:\n" "sub.u32 xa, spt, 16;\n" BGI_LDTM("x", "xa") BGI_WAITLD \
    "tcgen05.st.sync.aligned.32x32b.x16.b32 [xa], {" BGI_R16(BGI_A) "};\n" "tcgen05.wait::st.sync.aligned;\n" \
    BGI_NEXT BGI_K16(BGI_MOVX) BGI_DISPATCH \
    "L_SWAPM_%=:\n" BGI_GETM BGI_STM("ma", BGI_A) BGI_NEXT BGI_K16(BGI_MOVX) BGI_DISPATCH \
    BGI_PUSHES(KEEP) "L_KEEP_%=:\n" BGI_NEXT BGI_DISPATCH

#define BGI_HANDLERS \
    BGI_UNARY(SIN, BGI_SIN) BGI_UNARY(COS, BGI_COS) BGI_UNARY(LOG, BGI_LOG) BGI_UNARY(SQRT, BGI_SQRT) BGI_UNARY(EXP, BGI_EXP) \
    BGI_ENTRY_LX(SIN) BGI_ENTRY_LX(COS) BGI_ENTRY_LX(LOG) BGI_ENTRY_LX(SQRT) BGI_ENTRY_LX(EXP) \
    BGI_BIN_X(ADD, BGI_ADDX) BGI_ENTRY_S(ADD) BGI_ENTRY_M(ADD) BGI_ENTRY_LXX(ADD) \
    BGI_BIN_X(MUL, BGI_MULX) BGI_ENTRY_S(MUL) BGI_ENTRY_M(MUL) BGI_ENTRY_LXX(MUL) BGI_ENTRY_R \
    BGI_BIN_X(SUB, BGI_SUBX) BGI_ENTRY_LXX(SUB) \
    BGI_BIN_X(DIV, BGI_DIVX) BGI_ENTRY_LXX(DIV) \
    BGI_BIN_X(RSUB, BGI_RSUBX) BGI_ENTRY_S(RSUB) BGI_ENTRY_M(RSUB) \
    BGI_BIN_X(RDIV, BGI_RDIVX) BGI_ENTRY_S(RDIV) BGI_ENTRY_M(RDIV) \
    BGI_BIN_C(ADD, BGI_ADDC) BGI_BIN_C(SUB, BGI_SUBC) BGI_BIN_C(MUL, BGI_MULC) BGI_BIN_C(RSUB, BGI_RSUBC) BGI_BIN_C(RDIV, BGI_RDIVC) \
    BGI_ENTRY_LX(ADDC) BGI_ENTRY_LX(SUBC) BGI_ENTRY_LX(MULC) BGI_ENTRY_LX(RSUBC) BGI_ENTRY_LX(RDIVC) \
    BGI_PUSHES(LX) "L_LX_%=:\n" BGI_LXA BGI_NEXT BGI_WAITLD BGI_DISPATCH \
    BGI_PUSHES(LC) "L_LC_%=:\n" "mov.b32 cv, o;\n" BGI_NEXT BGI_K16(BGI_LC) BGI_DISPATCH \
    BGI_PUSHES(LS) "L_LS_%=:\n" "add.u32 xa, o, db;\n" BGI_NEXT \
    "ld.shared.v4.f32 {" BGI_A "0, " BGI_A "1, " BGI_A "2, " BGI_A "3}, [xa];\n" \
    "ld.shared.v4.f32 {" BGI_A "4, " BGI_A "5, " BGI_A "6, " BGI_A "7}, [xa+512];\n" \
    "ld.shared.v4.f32 {" BGI_A "8, " BGI_A "9, " BGI_A "10, " BGI_A "11}, [xa+1024];\n" \
    "ld.shared.v4.f32 {" BGI_A "12, " BGI_A "13, " BGI_A "14, " BGI_A "15}, [xa+1536];\n" BGI_DISPATCH \
    BGI_PUSHES(LG) "L_LG_%=:\n" "cvt.u64.u32 ma, o;\n" "add.u64 ma, ma, gb;\n" BGI_NEXT \
    "ld.global.nc.v4.f32 {" BGI_A "0, " BGI_A "1, " BGI_A "2, " BGI_A "3}, [ma];\n" \
    "ld.global.nc.v4.f32 {" BGI_A "4, " BGI_A "5, " BGI_A "6, " BGI_A "7}, [ma+512];\n" \
    "ld.global.nc.v4.f32 {" BGI_A "8, " BGI_A "9, " BGI_A "10, " BGI_A "11}, [ma+1024];\n" \
    "ld.global.nc.v4.f32 {" BGI_A "12, " BGI_A "13, " BGI_A "14, " BGI_A "15}, [ma+1536];\n" BGI_DISPATCH \
    BGI_UNARY(NEG, BGI_NEG) BGI_UNARY(SQR, BGI_SQRE) BGI_UNARY(CUBE, BGI_CUBE) \
    BGI_ENTRY_LX(NEG) BGI_ENTRY_LX(SQR) BGI_ENTRY_LX(CUBE) \
    BGI_STACKOPS

// ---- the dispatcher: the one indexed branch ----------------------------------------------------------------
#define BGI_DISPATCHER \
    "DISP_%=:\n" \
    "and.b32 hn, h, 255;\n" \
    "brx.idx.uni hn, TBL_%=;\n"

#define BGI_T(L) "L_" #L "_%=, "
#define BGI_TP(L) "P_" #L "_%=, "
#define BGI_TM(L) "M_" #L "_%=, "
#define BGI_FRESH(T) \
    T(LX) T(LC) T(LX_SIN) T(LX_COS) T(LX_LOG) T(LX_SQRT) T(LX_EXP) T(LX_NEG) T(LX_SQR) T(LX_CUBE) \
    T(LX_ADDX) T(LX_SUBX) T(LX_MULX) T(LX_DIVX) \
    T(LX_ADDC) T(LX_SUBC) T(LX_MULC) T(LX_RSUBC) T(LX_RDIVC) T(LX_MULR) T(LS) T(LG) T(KEEP)
#define BGI_TABLE \
    "TBL_%=: .branchtargets " \
    BGI_T(END) BGI_T(SIN) BGI_T(COS) BGI_T(LOG) BGI_T(SQRT) BGI_T(EXP) BGI_T(NEG) BGI_T(SQR) BGI_T(CUBE) \
    BGI_T(ADDX) BGI_T(SUBX) BGI_T(MULX) BGI_T(DIVX) BGI_T(RSUBX) BGI_T(RDIVX) \
    BGI_T(ADDS) BGI_T(MULS) BGI_T(RSUBS) BGI_T(RDIVS) \
    BGI_T(ADDM) BGI_T(MULM) BGI_T(RSUBM) BGI_T(RDIVM) \
    BGI_T(ADDC) BGI_T(SUBC) BGI_T(MULC) BGI_T(RSUBC) BGI_T(RDIVC) \
    BGI_T(MULR) BGI_T(POPS) BGI_T(POPM) BGI_T(SWAPS) BGI_T(SWAPM) \
    BGI_FRESH(BGI_T) BGI_FRESH(BGI_TP) BGI_FRESH(BGI_TM) \
    "L_END_%=;\n"

// ---- variant 1: one program, one pass; the accumulator is the asm's output operands %0..%15 ------------------
// Operands: %0..%15 = acc (used in place), %16 = shared address of the records, %17 = xb, %18 = sb, %19 = rb, %20 = db (this lane's
// shared-memory address of the staged unary rows of this pass), %21 = gb (the same in global memory).
#define BGI_ASM \
    "{\n" \
    ".reg .f32 x<16>, t<16>, q<16>, cv;\n" \
    ".reg .pred p<16>;\n" \
    ".reg .b32 h, o, hn, pc, xa, xb, rb, db, spt, e;\n" \
    ".reg .b64 ma, mbase, gb;\n" \
    ".local .align 16 .b8 slotmem[1984];\n"      /* kMemSlots * 64 */ \
    BGI_TABLE \
    "mov.u32 pc, %16;\n" \
    "mov.u32 xb, %17;\n" \
    "mov.u32 spt, %18;\n" \
    "mov.u32 rb, %19;\n" \
    "mov.u32 db, %20;\n" \
    "mov.u64 gb, %21;\n" \
    "mov.u64 mbase, slotmem;\n" \
    "ld.shared.v2.b32 {h, o}, [pc];\n" \
    BGI_DISPATCHER \
    BGI_HANDLERS \
    "L_END_%=:\n" \
    "}\n"

#define BGI_ACC_OUT(A) "=&f"(A[0]), "=&f"(A[1]), "=&f"(A[2]), "=&f"(A[3]), "=&f"(A[4]), "=&f"(A[5]), "=&f"(A[6]), "=&f"(A[7]), \
                       "=&f"(A[8]), "=&f"(A[9]), "=&f"(A[10]), "=&f"(A[11]), "=&f"(A[12]), "=&f"(A[13]), "=&f"(A[14]), "=&f"(A[15])

// ---- variant 2: a whole GROUP of programs, all passes, with a7 inside the block (MSE fitness) ----------------------
// The END record of a program carries what the frame around variant 1 read from the queue window: rec[n] = { H_END |
// stride << 8, p }, rec[n+1] = { (float)L, 0 } (k_compile). END is then a handler like the others: residual against y
// in the canonical order (DESIGN.md §7 "summation order"), next pass (the operand bases move on, the records are
// run again) or the butterfly, the mean, the length tax, the store of fitness[p]; the next program of the group starts
// `stride` records after the start of this one. One entry into the block per group instead of one per program and pass.
// Operands: %0 records of the group, %1 xb of pass 0, %2 sb, %3 rb of pass 0, %4 db of pass 0, %5 gb of pass 0,
// %6 this lane's address of y (float4 index lane of pass 0), %7 programs in the group, %8 passes, %9 / %10 columns per
// pass of the variable / reciprocal block, %11 = n - 4 * lane (a case k of 128-case block g of pass s counts when
// 512 s + 128 g + k < that), %12 = (float)n, %13 = 1 / n when n is a power of two (the mean is then an exact scaling,
// bit-identical to the division), else 0, %14 tax, %15 fitness, %16 != 0: this lane stores (lane 0), %17 = n.
// A call with more than 512 cases is SPLIT into one launch per pass (eval_kernel.inc): %18 = the lanes' parked sums
// (32 floats per individual), %19 = 0 one launch does everything, 1 the launch of pass 0 (parks the sums), 2 the launch
// of pass 1 (takes them back before its own residuals: the lane's chain of fma continues as if there had been one launch),
// %20 = 4 * lane.
#define BGI_SQ(k)   "sub.rn.f32 t" #k ", " BGI_A #k ", x" #k ";\n" "fma.rn.f32 sum, t" #k ", t" #k ", sum;\n"
#define BGI_SQR(k, LIM) "setp.lt.s32 p" #k ", " LIM ", nrem;\n" "sub.rn.f32 t" #k ", " BGI_A #k ", x" #k ";\n" "@p" #k " fma.rn.f32 sum, t" #k ", t" #k ", sum;\n"
#define BGI_BFLY(M) "shfl.sync.bfly.b32 cv, sum, " #M ", 0x1f, 0xffffffff;\n" "add.rn.f32 sum, sum, cv;\n"
#define BGI_LDY \
    "ld.shared.v4.f32 {x0, x1, x2, x3}, [ya];\n" \
    "ld.shared.v4.f32 {x4, x5, x6, x7}, [ya+512];\n" \
    "ld.shared.v4.f32 {x8, x9, x10, x11}, [ya+1024];\n" \
    "ld.shared.v4.f32 {x12, x13, x14, x15}, [ya+1536];\n"
#define BGI_END_GROUP \
    "L_END_%=:\n" \
    "setp.eq.u32 pr, %19, 2;\n"                   /* second launch of a split call: the lane's sum of pass 0 comes back */ \
    "@!pr bra.uni NOPART_%=;\n" \
    "mul.wide.u32 ma, o, 128;\n" "add.u64 ma, ma, %18;\n" "cvt.u64.u32 mb, %20;\n" "add.u64 ma, ma, mb;\n" \
    "ld.global.f32 sum, [ma];\n" \
    "NOPART_%=:\n" \
    BGI_LDY \
    "setp.lt.s32 pr, nleft, 512;\n"               /* a ragged last pass: the padded cases do not count */ \
    "@pr bra.uni RAG_%=;\n" \
    BGI_K16(BGI_SQ) \
    "bra.uni PASSED_%=;\n" \
    "RAG_%=:\n" \
    BGI_SQR(0, "0") BGI_SQR(1, "1") BGI_SQR(2, "2") BGI_SQR(3, "3") \
    BGI_SQR(4, "128") BGI_SQR(5, "129") BGI_SQR(6, "130") BGI_SQR(7, "131") \
    BGI_SQR(8, "256") BGI_SQR(9, "257") BGI_SQR(10, "258") BGI_SQR(11, "259") \
    BGI_SQR(12, "384") BGI_SQR(13, "385") BGI_SQR(14, "386") BGI_SQR(15, "387") \
    "PASSED_%=:\n" \
    "add.u32 ps, ps, 1;\n" \
    "setp.lt.u32 pr, ps, %8;\n" \
    "@!pr bra.uni FIN_%=;\n" \
    "add.u32 xb, xb, %9;\n" "add.u32 rb, rb, %10;\n" "add.u32 db, db, 2048;\n" "add.u64 gb, gb, 2048;\n" \
    "add.u32 ya, ya, 2048;\n" "sub.s32 nrem, nrem, 512;\n" "sub.s32 nleft, nleft, 512;\n" \
    "mov.u32 pc, pc0;\n" "mov.u32 spt, %2;\n" \
    "ld.shared.v2.b32 {h, o}, [pc];\n" \
    "bra.uni DISP_%=;\n" \
    "FIN_%=:\n" \
    "setp.eq.u32 pr, %19, 1;\n"                   /* first launch of a split call: park the lane's sum, no fitness yet */ \
    "@!pr bra.uni FINAL_%=;\n" \
    "mul.wide.u32 ma, o, 128;\n" "add.u64 ma, ma, %18;\n" "cvt.u64.u32 mb, %20;\n" "add.u64 ma, ma, mb;\n" \
    "st.global.f32 [ma], sum;\n" \
    "bra.uni NEXTP_%=;\n" \
    "FINAL_%=:\n" \
    "ld.shared.f32 q0, [pc+8];\n"                 /* (float)L */ \
    BGI_BFLY(16) BGI_BFLY(8) BGI_BFLY(4) BGI_BFLY(2) BGI_BFLY(1) \
    "setp.neu.f32 pr, %13, 0f00000000;\n" \
    "@pr bra.uni MEANM_%=;\n" \
    "div.rn.f32 sum, sum, %12;\n" \
    "bra.uni MEAND_%=;\n" \
    "MEANM_%=:\n" \
    "mul.rn.f32 sum, sum, %13;\n" \
    "MEAND_%=:\n" \
    "fma.rn.f32 sum, %14, q0, sum;\n" \
    "mul.wide.u32 ma, o, 4;\n" "add.u64 ma, ma, %15;\n" \
    "setp.ne.u32 pr, %16, 0;\n" \
    "@pr st.global.f32 [ma], sum;\n" \
    "NEXTP_%=:\n" \
    "sub.u32 gc, gc, 1;\n" \
    "setp.eq.u32 pr, gc, 0;\n" \
    "@pr bra.uni EXIT_%=;\n" \
    "shr.u32 e, h, 8;\n" "shl.b32 e, e, 3;\n" "add.u32 pc0, pc0, e;\n" "mov.u32 pc, pc0;\n" \
    "mov.u32 xb, %1;\n" "mov.u32 rb, %3;\n" "mov.u32 db, %4;\n" "mov.u64 gb, %5;\n" "mov.u32 ya, %6;\n" \
    "mov.u32 spt, %2;\n" "mov.s32 nrem, %11;\n" "mov.s32 nleft, %17;\n" "mov.u32 ps, 0;\n" "mov.f32 sum, 0f00000000;\n" \
    "ld.shared.v2.b32 {h, o}, [pc];\n" \
    "bra.uni DISP_%=;\n"

#define BGI_ASM_GROUP \
    "{\n" \
    ".reg .f32 a<16>, x<16>, t<16>, q<16>, cv, sum;\n" \
    ".reg .pred p<16>, pr;\n" \
    ".reg .b32 h, o, hn, pc, pc0, xa, xb, rb, db, spt, e, ya, gc, ps;\n" \
    ".reg .s32 nrem, nleft;\n" \
    ".reg .b64 ma, mb, mbase, gb;\n" \
    ".local .align 16 .b8 slotmem[1984];\n" \
    BGI_TABLE \
    "mov.u32 pc, %0;\n" "mov.u32 pc0, %0;\n" \
    "mov.u32 xb, %1;\n" "mov.u32 spt, %2;\n" "mov.u32 rb, %3;\n" "mov.u32 db, %4;\n" "mov.u64 gb, %5;\n" \
    "mov.u32 ya, %6;\n" "mov.u32 gc, %7;\n" "mov.s32 nrem, %11;\n" "mov.s32 nleft, %17;\n" "mov.u32 ps, 0;\n" "mov.f32 sum, 0f00000000;\n" \
    "mov.u64 mbase, slotmem;\n" \
    "ld.shared.v2.b32 {h, o}, [pc];\n" \
    BGI_DISPATCHER \
    BGI_HANDLERS \
    BGI_END_GROUP \
    "EXIT_%=:\n" \
    "}\n"

namespace beagle {

static_assert(kMemSlots * 64 == 1984 && kCasesPerLane == 16, "interp.cuh is written for 16 cases per lane and 31 memory slots");
static_assert(H_COUNT == 102 && H_KEEP == H_FRESH0 + H_NFRESH - 1, "BGI_TABLE lists the handlers in the order of uop.cuh's enum");

// acc[k] = the program's output on case (pass * 512 + (k/4)*128 + lane*4 + k%4)
#define BGI_A "%"
__device__ __forceinline__ void interp_run(uint32_t rec, uint32_t xb, uint32_t sb, uint32_t rb, uint32_t db, const float* gb, float (&acc)[16])
{
    asm volatile(BGI_ASM : BGI_ACC_OUT(acc) : "r"(rec), "r"(xb), "r"(sb), "r"(rb), "r"(db), "l"(gb) : "memory");
}
#undef BGI_A

// a group of `count` programs whose record blocks follow one another from `rec` on, every pass, fitness[p] stored
struct GroupArgs {
    uint32_t xb, sb, rb, db; const float* gb; uint32_t ya; uint32_t passes, xstride, rstride; int nrem;
    float nf, inv_n, tax; float* fitness; uint32_t lane0; int n; float* partial; uint32_t lane4;
};
#define BGI_A "a"
template <int PMODE>                               // an immediate: ptxas folds the two tests of the END handler away
__device__ __forceinline__ void interp_group(uint32_t rec, uint32_t count, const GroupArgs& g)
{
    asm volatile(BGI_ASM_GROUP :: "r"(rec), "r"(g.xb), "r"(g.sb), "r"(g.rb), "r"(g.db), "l"(g.gb), "r"(g.ya), "r"(count),
                 "r"(g.passes), "r"(g.xstride), "r"(g.rstride), "r"(g.nrem), "f"(g.nf), "f"(g.inv_n), "f"(g.tax), "l"(g.fitness),
                 "r"(g.lane0), "r"(g.n), "l"(g.partial), "n"(PMODE), "r"(g.lane4) : "memory");
}
#undef BGI_A

} // namespace beagle
