// ucode.h - the lowered program format of the bit-sliced kernel (host lowering <-> device kernel).
//
// A postfix program (include/kripke.h opcodes) is lowered on the host (lower.cpp) to a straight
// sequence of 16-bit micro-ops (low byte = op, high byte = argument) over a register stack of at
// most UC_DMAX slots D0..D3.  Every micro-op names its slot statically, so the kernel keeps the
// whole stack in registers (the paper's 48-slot stack went to 272 B of thread-local memory,
// PAPER.md:72).  What the lowering removes before the kernel ever runs:
//   * negation: a polarity bit per value is folded into the next operator (De Morgan, box/dia
//     duality); constants are folded;
//   * pushes of atoms: an atom that is an operand of a binary connective is read directly by the
//     connective's micro-op (BOOLV / BOOLL), it never occupies a slot;
//   * modal operators applied to a constant or to the in-word variable p_0: box F ("dead end"),
//     dia T, box p_0, dia p_0 (and their negations) depend on the frame only, so the kernel computes
//     them once per scan unit as "derived leaves" and every program reads them like atoms.
//   * loads that feed the next operator directly (LOWER_FUSE): "load q; box" becomes one micro-op
//     that reads q where it lives - one dispatch and one register copy fewer, and the compile-time
//     bits of q fold into the logic;
// The last micro-op is one of the FIN ops and produces, per 32-model word, the mask of models that
// refute the formula (or distinguish the pair).
#pragma once
#include <stdint.h>

namespace kripke {

constexpr int UC_DMAX = 4;       // register-stack slots

// leaves read from the per-thread leaf table (argument byte of LOADL / BOOLL)
enum : uint8_t { LEAF_P = 0, LEAF_DEAD = 1, LEAF_BOXP = 2, LEAF_DIAP = 3, LEAF_COUNT = 4 };

// lowering modes (which derived leaves the target kernel instantiation provides)
enum : uint32_t {
    LOWER_LEAF_DEAD = 1u << 0,   // box F / dia T as a leaf
    LOWER_LEAF_P = 1u << 1,      // p_0, box p_0, dia p_0 as leaves (p_0 lies inside the 32-model word)
    LOWER_FUSE = 1u << 2         // fold a load into the modal operator that follows it (fused ops below)
};

// Boolean functions of (slot value a, operand b); the lowering picks one by the two polarities
enum : uint8_t { BF_AND = 0, BF_OR = 1, BF_ANDN = 2 /* a & ~b */, BF_NAND = 3 /* ~a & b */ };

enum : uint8_t {
    UC_LOADV = 0,     // + i*4 + d          : D[d] <- p_i
    UC_BOOLV = 16,    // + (f*4 + i)*4 + d  : D[d] <- f(D[d], p_i)
    UC_LOADL = 80,    // + d   (arg = leaf) : D[d] <- leaf
    UC_BOOLL = 84,    // + f*4 + d (arg = leaf) : D[d] <- f(D[d], leaf)
    UC_BOOL = 100,    // + f*4 + d          : D[d] <- f(D[d], D[d+1])        (d = 0..2)
    UC_BOX = 116,     // + d                : D[d] <- box D[d]
    UC_DIA = 120,     // + d                : D[d] <- dia D[d]
    UC_FIN_ALL = 124, // refuted = ~(D0[0] & ... & D0[n-1])      truth set = D0
    UC_FIN_ANY = 125, // refuted =   D0[0] | ... | D0[n-1]       truth set = ~D0
    UC_FIN_XOR = 126, // differ  = OR_w (D0[w] ^ D1[w])          pair, equal polarities
    UC_FIN_XNOR = 127,// differ  = OR_w ~(D0[w] ^ D1[w])         pair, opposite polarities
    UC_LOADZ = 128,   // + d                : D[d] <- all-false
    // fused forms (LOWER_FUSE): the operand is read where it lives instead of being loaded first
    UC_BOXV0 = 132,   // + i                : D[0] <- box p_i
    UC_DIAV0 = 136,   // + i                : D[0] <- dia p_i
    UC_BOXL = 140,    // + d   (arg = leaf) : D[d] <- box leaf
    UC_DIAL = 144     // + d   (arg = leaf) : D[d] <- dia leaf
};

}  // namespace kripke
