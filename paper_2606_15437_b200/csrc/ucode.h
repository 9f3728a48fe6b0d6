// ucode.h - the lowered program format of the bit-sliced kernel (host lowering <-> device kernel).
//
// A postfix program (include/kripke.h opcodes) is lowered on the host (lower.cpp) to a straight
// sequence of one-byte micro-ops over a register stack of DMAX slots D0..D3.  Every micro-op names
// its slot statically, so the kernel keeps the whole stack in registers (the paper's 48-slot stack
// went to 272 B of thread-local memory).  Negation never executes: the lowering tracks
// a polarity bit per slot and folds it into the next operator (De Morgan / box-dia duality), and
// constants are folded.  The last micro-op is one of the FIN ops and produces, per 32-model word,
// the mask of models that refute the formula (or distinguish the pair).
#pragma once
#include <stdint.h>

namespace kripke {

constexpr int UC_DMAX = 4;       // register-stack slots
constexpr int UC_NATOMS = 5;     // p0..p3 and the all-false constant

enum : uint8_t {
    UC_PUSH = 0,      // + atom * UC_DMAX + d : D[d] <- atom      (atom 0..3 = p_i, 4 = all-false)
    UC_BOX = 20,      // + d : D[d] <- box D[d]
    UC_DIA = 24,      // + d : D[d] <- dia D[d]
    UC_AND = 28,      // + d : D[d] <- D[d] & D[d+1]       (d = 0..2)
    UC_OR = 31,       // + d : D[d] <- D[d] | D[d+1]
    UC_ANDN = 34,     // + d : D[d] <- D[d] & ~D[d+1]
    UC_NAND = 37,     // + d : D[d] <- ~D[d] & D[d+1]
    UC_FIN_ALL = 40,  // refuted = ~(D0[0] & ... & D0[n-1])      truth set = D0
    UC_FIN_ANY = 41,  // refuted =   D0[0] | ... | D0[n-1]       truth set = ~D0
    UC_FIN_XOR = 42,  // differ  = OR_w (D0[w] ^ D1[w])          pair, equal polarities
    UC_FIN_XNOR = 43, // differ  = OR_w ~(D0[w] ^ D1[w])         pair, opposite polarities
    UC_COUNT = 44
};

}  // namespace kripke
