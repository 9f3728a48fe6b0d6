// wf_ucode.h - lowered program format of the warp-frame kernel (scan_wf.cuh), host lowering <->
// device kernel.
//
// In the warp-frame layout one warp evaluates a program on a group of 2^MB "sibling" frames at a
// time: the frames of a group differ only in MB edge bits of one row w0 of the relation (the
// "m-row"); every valuation of the group's frames lies in the 32 lanes x 32 word bits (plus, for
// fewer variables, more frame bits).  A subformula of modal depth 0 does not depend on the frame at
// all, and one of modal depth 1 depends on the sibling index only at world w0.  The lowering
// therefore types every value by its modal depth:
//     S  (depth 0)   n words, shared by all 2^MB siblings
//     H  (depth 1)   n-1 shared words + 2^MB words for world w0
//     F  (depth >=2) 2^MB x n words
// and every micro-op names the typed registers it reads and writes, so all values stay in
// registers and work that is the same for all siblings is done once (Proposition 1:
// the cost of a formula is |phi| + d*n word operations per model - here per *distinct* word).
//
// Stack discipline (lower.cpp, WfLowerer): of the two operands of a binary connective the one of
// higher type is evaluated first; hence, when an operand of lower type is evaluated, no value of
// its type is pending, and it always lands in slot 0 of its type.  That keeps the number of
// register-naming variants per micro-op small:
//     S values: slots S0..S3 (stack)      H values: H0, H1 (stack)      F values: buffers F0, F1
// A modal operator on an F value writes the other F buffer (it needs all worlds of its operand
// until the last row is done), so only one F value can be live: a program that needs two is left
// to the bit-sliced kernel.
//
// Negation never executes (polarity folding, as in ucode.h); constants are folded.
#pragma once
#include <stdint.h>

namespace kripke {

// atom argument (high byte) of LOADA / B?A: 0 = the constant false, 1 + i = variable p_i
enum : uint8_t { WF_ATOM_FALSE = 0, WF_ATOM_VAR0 = 1 };

// Boolean functions: same numbering as ucode.h (BF_AND, BF_OR, BF_ANDN a&~b, BF_NAND ~a&b); the
// first operand is the value already in the destination.
// t = 0 box, 1 dia.   pol = 0: the value is the truth set, 1: its complement.
enum : uint8_t {
    WF_LOADA = 0,    // + d            (4)  S[d] <- atom(arg)
    WF_BSA = 4,      // + f*4 + d     (16)  S[d] <- f(S[d], atom(arg))
    WF_BSS = 20,     // + f*4 + d     (16)  S[d] <- f(S[d], S[d+1])            d = 0..2
    WF_S2H = 36,     // + t*2 + h      (4)  H[h] <- modal_t(S[0])
    WF_BHA = 40,     // + f*2 + h      (8)  H[h] <- f(H[h], atom(arg))
    WF_BHS = 48,     // + f*2 + h      (8)  H[h] <- f(H[h], S[0])
    WF_BHH = 56,     // + f            (4)  H[0] <- f(H[0], H[1])
    WF_H2F = 60,     // + t*2 + b      (4)  F[b] <- modal_t(H[0])
    WF_MF = 64,      // + t*2 + b      (4)  F[1-b] <- modal_t(F[b])
    WF_BFA = 68,     // + f*2 + b      (8)  F[b] <- f(F[b], atom(arg))
    WF_BFS = 76,     // + f*2 + b      (8)  F[b] <- f(F[b], S[0])
    WF_BFH = 84,     // + f*2 + b      (8)  F[b] <- f(F[b], H[0])
    WF_FIN_S = 92,   // + pol          (2)  refuted = S[0] is not all worlds
    WF_FIN_H = 94,   // + pol          (2)  ... H[0]
    WF_FIN_F = 96,   // + pol*2 + b    (4)  ... F[b]
    WF_OP_COUNT = 100
};

constexpr int WF_S_SLOTS = 4, WF_H_SLOTS = 2;

// Per-launch capacity: the programs travel in the kernel parameter block (constant bank, read
// through the uniform datapath), which is limited to 32,764 bytes.
constexpr uint32_t WF_MAX_PROGS = 1024;
constexpr uint32_t WF_MAX_UCODE = 12288;

// What a lowered program costs, in micro-ops of each cost class (the kernel shape turns these into
// instruction counts: see wf_cost in scan_wf_inst.cu).
struct WfOpCounts {
    uint32_t bool_s = 0, bool_h = 0, bool_f = 0;     // Boolean micro-ops by result type
    uint32_t modal_s = 0, modal_hf = 0;              // modal micro-ops by operand type (S ; H or F)
    uint32_t fin_type = 0;                           // 0 S, 1 H, 2 F
};

}  // namespace kripke
