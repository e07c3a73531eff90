// uop.cuh — the micro-op stream between the tree compiler (k_compile, a3/a5) and the interpreter
// (k_eval_*, a6). DESIGN.md §7.
//
// A Beagle program is postfix, i.e. a tree. The compiler turns it into code for an
// ACCUMULATOR machine: `acc` (K cases per lane, in registers) holds the most recently computed
// value, s[0..D) hold computed values that wait for their sibling. Terminals (CONST, LOAD) that are
// the operand of a binary command are folded into that command, so they cost no dispatch and no
// register move:
//     a x  ADD     ->  ADDX x        acc = acc + X[x]          (right operand terminal)
//     x <A> SUB    ->  XSUB x        acc = X[x] - acc          (left operand terminal)
//     <A> <B> DIV  ->  ... PUSH ... DIVS S   acc = s[S] / acc  (both computed)
// Every micro-op computes exactly the value the postfix command computes on the same operands with
// the same per-command function (ops.cuh), so per-case outputs are bit-identical to a plain stack
// machine; only the ORDER in which independent subtrees are evaluated may differ (Sethi-Ullman:
// the subtree that needs more slots first), which no result depends on.
//
// Encoding: uint2 {x = handler | operand << 8, y = literal}. operand = byte offset of the variable's
// row in the staged case block (LOAD-type), literal = the fp32 constant's bits (CONST-type).
// Handler numbers are dense so that the interpreter's switch is one jump table.
#pragma once
#include <stdint.h>

namespace beagle {

constexpr int kSlotsMax = 8;   // s[] slots any program of <= 512 tokens can need is <= 7

enum : uint32_t {
    H_END = 0,
    H_LOADX = 1, H_CONST = 2,                                  // acc = X[j] | c      (acc was dead)
    H_SIN = 3, H_COS = 4, H_LOG = 5, H_SQRT = 6, H_EXP = 7,    // acc = f(acc)
    H_ADDX = 8, H_SUBX = 9, H_MULX = 10, H_DIVX = 11,          // acc = acc op X[j]
    H_XSUB = 12, H_XDIV = 13,                                  // acc = X[j] op acc
    H_ADDC = 14, H_SUBC = 15, H_MULC = 16, H_DIVC = 17,        // acc = acc op c
    H_CSUB = 18, H_CDIV = 19,                                  // acc = c op acc
    H_PUSHX = 20,                                              // +S: s[S] = acc; acc = X[j]
    H_PUSHC = H_PUSHX + kSlotsMax,                             // +S: s[S] = acc; acc = c
    H_ADDS = H_PUSHC + kSlotsMax,                              // +S: acc = s[S] + acc
    H_SUBS = H_ADDS + kSlotsMax,                               // +S: acc = s[S] - acc
    H_MULS = H_SUBS + kSlotsMax,                               // +S: acc = s[S] * acc
    H_DIVS = H_MULS + kSlotsMax,                               // +S: acc = s[S] / acc
    H_RSUBS = H_DIVS + kSlotsMax,                              // +S: acc = acc - s[S]
    H_RDIVS = H_RSUBS + kSlotsMax,                             // +S: acc = acc / s[S]
    H_COUNT = H_RDIVS + kSlotsMax
};

// meta[i] (one int4 per individual, in evaluation order): x = p (input index), y = uop block address
// in 16-byte units, z = nu | slots << 16 | kind << 24, w = length in tokens (for the tax).
enum : int { KIND_MAIN = 0, KIND_DEEP = 1, KIND_SKIP = 2 };

} // namespace beagle
