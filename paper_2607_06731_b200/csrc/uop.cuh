// uop.cuh — the micro-op stream between the tree compiler (k_compile, a3/a5) and the interpreter
// (k_eval, a6). DESIGN.md §7.
//
// A Beagle program is postfix, i.e. a tree. The compiler turns it into code for an
// ACCUMULATOR machine: `acc` (16 cases per lane, in registers) holds the most recently computed
// value; s[0], s[1], ... hold computed values that wait for their sibling (s[0..kRegSlots) in
// registers, the rest in local memory: "spilling only when needed"). Terminals (CONST, LOAD) that are
// the operand of a binary command are folded into that command, so they cost no dispatch and no
// register move:
//     <A> x  ADD     ->  ADDX x        acc = acc + X[x]          (right operand terminal)
//     x <A> SUB      ->  XSUB x        acc = X[x] - acc          (left operand terminal)
//     <A> <B> DIV    ->  ... PUSH S ... DIVS S   acc = s[S] / acc  (both computed)
// Commands run in the program's own order, and every micro-op computes exactly the value the postfix
// command computes on the same operands with the same per-command function (ops.cuh / interp.cuh), so
// per-case outputs are bit-identical to a plain stack machine (ADD and MUL commute bit for bit).
//
// Stream layout (uint2 records, one TMA bulk copy per program): the handler number of micro-op j+1
// travels in record j, so that when handler j starts, the jump-table index of its successor is already
// in a register and the table lookup overlaps the handler's arithmetic:
//     rec[0]   = { handler_0,                      0         }
//     rec[j+1] = { handler_{j+1} | extra_j << 8,   operand_j }      j = 0 .. n-1, handler_n = H_END
//     rec[n+1] = { H_END, 0 }                                        (prefetch pad)
// operand_j: byte offset of the variable's row in the staged case block (X-type), the fp32 constant's
// bits (C-type); extra_j: byte offset of the slot in the lane's local slot memory (M-type).
#pragma once
#include <stdint.h>

namespace beagle {

constexpr int kRegSlots = 4;    // s[0..4) live in registers
constexpr int kMemSlots = 27;   // s[4..31) live in local memory (a 32-entry stack pushes at most 31 values)

enum : uint32_t {
    H_END = 0,
    H_LOADX = 1, H_CONST = 2,                                  // acc = X[j] | c      (acc was dead)
    H_SIN = 3, H_COS = 4, H_LOG = 5, H_SQRT = 6, H_EXP = 7,    // acc = f(acc)
    H_ADDX = 8, H_SUBX = 9, H_MULX = 10, H_DIVX = 11,          // acc = acc op X[j]
    H_XSUB = 12, H_XDIV = 13,                                  // acc = X[j] op acc
    H_ADDC = 14, H_SUBC = 15, H_MULC = 16, H_DIVC = 17,        // acc = acc op c
    H_CSUB = 18, H_CDIV = 19,                                  // acc = c op acc
    H_PUSHX = 20,                                              // +S: s[S] = acc; acc = X[j]
    H_PUSHC = H_PUSHX + kRegSlots,                             // +S: s[S] = acc; acc = c
    H_ADDS = H_PUSHC + kRegSlots,                              // +S: acc = s[S] + acc
    H_SUBS = H_ADDS + kRegSlots,                               // +S: acc = s[S] - acc
    H_MULS = H_SUBS + kRegSlots,                               // +S: acc = s[S] * acc
    H_DIVS = H_MULS + kRegSlots,                               // +S: acc = s[S] / acc
    H_PUSHXM = H_DIVS + kRegSlots,                             // mem[extra] = acc; acc = X[j]
    H_PUSHCM = H_PUSHXM + 1,                                   // mem[extra] = acc; acc = c
    H_ADDM = H_PUSHXM + 2, H_SUBM = H_PUSHXM + 3, H_MULM = H_PUSHXM + 4, H_DIVM = H_PUSHXM + 5,   // acc = mem[extra] op acc
    H_COUNT = H_PUSHXM + 6
};

// meta[i] (one int4 per individual, in evaluation order): x = p (input index), y = record block address
// in 16-byte units, z = number of records to copy (even), w = length in tokens (for the tax);
// z == 0: nothing to evaluate (malformed, or handed to the slow path).

} // namespace beagle
