// frames.cuh - step H2 (frame enumerator + class filter) and the scalar recurrence of section 3.
// Device-only helpers shared by the kernels of this library.
#pragma once
#include <stdint.h>

#include "../../include/kripke.h"

namespace kripke {

// Class T (reflexive frames): the compact index c has n*(n-1) bits, the off-diagonal edge bits in
// ascending position; the frame index is c with a 1 inserted at every diagonal position w*n+w.
// Ascending c <=> ascending f, so class order is preserved.
__device__ __forceinline__ uint64_t reflexive_deposit(uint32_t n, uint64_t c) {
    uint64_t f = 0;
    const uint32_t rowbits = n - 1;
    const uint64_t rowmask = (1ull << rowbits) - 1;
    for (uint32_t w = 0; w < n; ++w) {
        uint64_t row = (c >> (w * rowbits)) & rowmask;
        uint64_t low = row & ((1ull << w) - 1);
        uint64_t high = row >> w;
        f |= (low | (1ull << w) | (high << (w + 1))) << (w * n);
    }
    return f;
}

// Class-order index -> K-index f ("constrained classes by relational filtering").
__device__ __forceinline__ uint64_t class_frame(uint32_t n, uint32_t cls, const uint64_t *table, uint64_t c) {
    if (cls == KRIPKE_CLASS_K) return c;
    if (cls == KRIPKE_CLASS_T) return reflexive_deposit(n, c);
    return table[c];
}

// The bitwise recurrence on one model: a world set is an n-bit mask, box/dia are
// Lemma 1's containment / intersection tests per world.  Postfix program, stack in local memory
// (this is the paper's own kernel layout; the bit-sliced kernel replaces it on the hot path).
__device__ inline uint32_t eval_postfix_scalar(const uint8_t *__restrict__ code, uint32_t len, uint32_t n,
                                               const uint32_t *succ, const uint32_t *val, uint32_t full) {
    uint32_t st[KRIPKE_MAX_STACK];
    int sp = 0;
    for (uint32_t pc = 0; pc < len; ++pc) {
        const uint32_t c = code[pc];
        if (c == KRIPKE_OP_TOP) st[sp++] = full;
        else if (c == KRIPKE_OP_BOT) st[sp++] = 0u;
        else if (c < KRIPKE_OP_NOT) st[sp++] = val[c - KRIPKE_OP_VAR0];
        else if (c == KRIPKE_OP_NOT) st[sp - 1] = full & ~st[sp - 1];
        else if (c == KRIPKE_OP_BOX) {
            const uint32_t x = st[sp - 1];
            uint32_t r = 0;
            for (uint32_t w = 0; w < n; ++w) r |= (uint32_t)((succ[w] & ~x) == 0u) << w;   // eq. (1)
            st[sp - 1] = r;
        } else if (c == KRIPKE_OP_DIA) {
            const uint32_t x = st[sp - 1];
            uint32_t r = 0;
            for (uint32_t w = 0; w < n; ++w) r |= (uint32_t)((succ[w] & x) != 0u) << w;    // eq. (2)
            st[sp - 1] = r;
        } else {
            const uint32_t y = st[--sp], x = st[sp - 1];
            st[sp - 1] = (c == KRIPKE_OP_AND) ? (x & y) : (c == KRIPKE_OP_OR) ? (x | y) : ((full & ~x) | y);
        }
    }
    return st[0];
}

}  // namespace kripke
