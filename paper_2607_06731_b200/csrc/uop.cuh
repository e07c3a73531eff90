// uop.cuh — the micro-op stream between the tree compiler (k_compile, a3/a5) and the interpreter
// (k_eval, a6). DESIGN.md §7.
//
// A Beagle program is postfix, i.e. a tree. The compiler turns it into code for an
// ACCUMULATOR machine: `acc` (16 cases per lane, in registers) holds the most recently computed
// value; computed values that wait for their sibling are pushed to slots. Slots are not registers:
// slot s < S_T lives in TENSOR MEMORY (16 columns of the warp's own TMEM lanes, written by one
// tcgen05.st and read back by one tcgen05.ld straight into the operand registers), deeper slots in
// local memory ("spilling only when needed"). The fitness-case matrix X lives in tensor memory too,
// so a variable operand and a slot operand are the same instruction with a different column.
//
// Terminals (CONST, LOAD) never cost a dispatch: they are folded into the command that consumes them,
//     <A> x  ADD     ->  ADDX  x          acc = acc + X[x]           (right operand terminal)
//     x <A> SUB      ->  RSUBX x          acc = X[x] - acc           (left operand terminal)
//     x  y  DIV      ->  LX_DIVX x, y     acc = X[x] / X[y]          (both terminal: a fresh value)
//     x  SIN         ->  LX_SIN x         acc = sin X[x]
//     <A> <B> DIV    ->  RDIVS s          acc = slot[s] / acc        (both computed)
//     x  SIN         ->  LS row           acc = (sin X[x]) staged once per CTA, when the row fits shared memory
//     <A> x  DIV     ->  MULR  x          acc = acc * (1/X)[x]       (division by a variable is loop-invariant:
//                                         when no case of x is protected, its reciprocals are a staged row)
// and "push acc" is not a micro-op either: the micro-op that starts the next fresh value is dispatched to
// the push entry of its handler (handler number + H_PUSHT or + H_PUSHM).
// Commands run in the program's own order and every micro-op computes exactly the value the postfix
// command computes on the same operands with the same per-command function (ops.cuh / interp.cuh), so
// per-case outputs are bit-identical to a plain stack machine (ADD and MUL commute bit for bit;
// x / c with a constant c is x * rcp(c) with the same rcp the division handler uses).
//
// Stream layout: uint2 records {h, o}, one per micro-op, one TMA bulk copy per program:
//     rec[j] = record of micro-op j,  j = 0 .. n-1;   rec[n] = { H_END, 0 };   rec[n+1] = pad
//   h  [7:0]    handler number (uop.cuh enum; fresh values: + H_PUSHT / + H_PUSHM when acc is pushed first)
//      [20:10]  H_PUSHM entries: local byte offset of the slot (slot * 64)
//      [31:21]  column of the FIRST operand of an LX_ micro-op (a variable: (pass-relative) column)
//   o           second operand: column of a variable (X-type), byte offset of a slot in local memory
//               (M-type), fp32 bits of a constant (C-type); S-type pops the tensor-memory slot stack
#pragma once
#include <stdint.h>

namespace beagle {

constexpr int kCasesPerLane = 16;          // K: cases per lane per pass (one pass = 512 cases)
constexpr int kCasesPerPass = 32 * kCasesPerLane;
constexpr int kTmemCols = 512;             // tensor memory columns of one SM (32-bit cells x 128 lanes)
constexpr int kMemSlots = 31;              // a 32-entry stack pushes at most 31 computed values

enum : uint32_t {
    H_END = 0,
    // acc = f(acc)                                (NEG SQR CUBE: GCL's SIGN SQUARE CUBE)
    H_SIN = 1, H_COS = 2, H_LOG = 3, H_SQRT = 4, H_EXP = 5, H_NEG = 6, H_SQR = 7, H_CUBE = 8,
    // acc = acc op X[o] | X[o] op acc            (x <- tensor memory, variable column)
    H_ADDX = 9, H_SUBX = 10, H_MULX = 11, H_DIVX = 12, H_RSUBX = 13, H_RDIVX = 14,
    // acc = slot op acc                          (x <- tensor memory, slot column)
    H_ADDS = 15, H_MULS = 16, H_RSUBS = 17, H_RDIVS = 18,
    // acc = slot op acc                          (x <- local memory)
    H_ADDM = 19, H_MULM = 20, H_RSUBM = 21, H_RDIVM = 22,
    // acc = acc op c | c op acc
    H_ADDC = 23, H_SUBC = 24, H_MULC = 25, H_RSUBC = 26, H_RDIVC = 27,
    H_MULR = 28,                                // acc = acc * (1 / X)[o]
    // GCL's stack commands on computed values: DEL of the top computed value, SWAP of the two topmost ones
    H_POPS = 29, H_POPM = 30,                   // acc = slot (tensor memory: the top of the slot stack | local memory at byte offset o)
    H_SWAPS = 31, H_SWAPM = 32,                 // acc <-> slot
    // fresh values: acc = X[colA] (then the command)
    H_LX = 33, H_LC = 34,                                             // acc = X[colA] | acc = c
    H_LX_SIN = 35, H_LX_COS = 36, H_LX_LOG = 37, H_LX_SQRT = 38, H_LX_EXP = 39, H_LX_NEG = 40, H_LX_SQR = 41, H_LX_CUBE = 42,
    H_LX_ADDX = 43, H_LX_SUBX = 44, H_LX_MULX = 45, H_LX_DIVX = 46,
    H_LX_ADDC = 47, H_LX_SUBC = 48, H_LX_MULC = 49, H_LX_RSUBC = 50, H_LX_RDIVC = 51,
    H_LX_MULR = 52,                             // acc = X[colA] * (1 / X)[o]: division by a variable whose reciprocal row is staged
    H_LS = 53,                                  // acc = F[o]: a staged row of f(X[j]) in shared memory (f unary, loop-invariant)
    H_LG = 54,                                  // acc = F[o]: the same row read from global memory (L2) when shared memory is full
    H_KEEP = 55,                                // acc = acc: with its push entry, DUP of a computed value (the copy goes to a slot)
    H_FRESH0 = H_LX, H_NFRESH = 23,             // the fresh-value handlers H_LX .. H_KEEP
    H_PUSHT = H_NFRESH,                         // + handler: push acc to the tensor-memory slot stack first
    H_PUSHM = 2 * H_NFRESH,                     // + handler: push acc to the local slot at byte offset h[20:10] first
    H_COUNT = H_FRESH0 + 3 * H_NFRESH
};

constexpr int kPushShift = 10, kColAShift = 21;

// meta[i] (one int4 per individual, in evaluation order): x = p (input index), y = record block address
// in 16-byte units, z = number of records to copy (even), w = length in tokens (for the tax);
// z == 0: nothing to evaluate (malformed, or handed to the slow path).

} // namespace beagle
