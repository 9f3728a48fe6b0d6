// scan_sliced.cuh - the hot path: bit-sliced fused corpus scan (steps H1-H7 of DESIGN.md).
//
// Layout.  The models of a class-K scan are numbered X = (f << k*n) | v.  A 32-bit word holds one
// truth bit for 32 consecutive models, so a truth set is N words (word w = "is world w in the set",
// for 32 models at once): this is the SWAR packing of BASELINE.json's north_star taken to 32 models
// per word.  Every connective of the recurrence becomes lane-wise logic:
//     and/or/imp : N   3-input logic instructions per 32 models
//     box        : R[w] = AND_u ( T[u] | ~E[w][u] )      N*N instructions      (Lemma 1, eq. 1)
//     dia        : R[w] = OR_u  ( T[u] &  E[w][u] )      N*N instructions      (Lemma 1, eq. 2)
// where E[w][u] is the word of edge bits w->u and atoms are words of valuation bits.  Because the
// model index is enumerated, those words are never loaded: index bits 0..4 vary inside the word
// and are the constants 0xAAAAAAAA, 0xCCCCCCCC, ... ; bits 5..5+MB-1 select one of the M = 2^MB
// words a thread holds (compile-time all-0 / all-1) ; all higher bits are thread-uniform masks
// decoded once per scan unit (steps H2, H3).  No frame array, valuation array or truth tensor
// exists.
//
// A thread evaluates a lowered program (ucode.h) on M words at a time; the register stack
// D[slot][m][w] lives entirely in registers because every micro-op names its slot statically.  The
// micro-op byte is warp-uniform, so the dispatch branch never diverges.
//
// Scan units.  If k*n >= 5+MB ("frame per unit") a unit is one class frame and the thread runs
// 2^(k*n-5-MB) passes over the valuation words of that frame; the frame's edge masks come from the
// class enumerator (K: identity, T: diagonal deposit, S4/S5: table), so all four classes run here.
// Otherwise ("group per unit", class K only) a unit is a group of 32*M consecutive models spanning
// 2^(5+MB-k*n) frames, and the low edge bits are the in-word / per-word constants.
//
// Reduction (step H6).  Per (unit, program): popcount of the refuting-lane words; per warp
// __ballot_sync / __reduce_add_sync; one shared-memory atomic triple per (warp, program); at the end
// of a work item one global atomic triple per (block, program) - the paper's block reduction
// with the warp step in between.  The first refuting frame is tracked as a minimum;
// the finish kernel (scan_scalar.cu) turns it into the (f, v, world) certificate.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "frames.cuh"
#include "internal.h"

namespace kripke {


struct SlicedParams {
    uint32_t cls;
    const uint64_t *class_table;
    uint64_t unit_begin;            // first scan unit
    uint64_t unit_count;
    const uint16_t *ucode;          // n_slots * stride micro-ops
    const uint32_t *slot_record;
    uint32_t n_slots;
    uint32_t stride;                // micro-ops per slot (even)
    uint32_t chunk;                 // slots per work item
    uint32_t n_chunks;
    uint32_t tiles_per_item;        // tiles of TPB (threads per block) units per work item
    uint32_t n_ranges;              // work items = n_ranges * n_chunks
    uint32_t model_shift;           // models count x 2^model_shift: variables the programs do not mention
    Accum *accum;
};

template <int N_, int K_, int MB_, int DMAX_>
struct SlicedCfg {
    static constexpr int N = N_, K = K_, MB = MB_;
    static constexpr int DMAX = DMAX_;                        // register-stack slots kept (<= UC_DMAX)
    static constexpr int M = 1 << MB;
    static constexpr int KN = K * N;
    static constexpr int LOW = 5 + MB;                        // index bits inside a thread's group
    static constexpr bool FRAME_PER_UNIT = KN >= LOW;
    static constexpr int PASS_BITS = FRAME_PER_UNIT ? KN - LOW : 0;
    static constexpr int UNIT_FRAME_BITS = FRAME_PER_UNIT ? 0 : LOW - KN;   // log2 frames per unit
    // p_0 lies entirely inside the 32-model word and the frame is thread-uniform: p_0, box p_0 and
    // dia p_0 are the same N words for every word the thread holds -> leaf-table entries
    static constexpr bool P_LEAF = FRAME_PER_UNIT && K >= 1 && N <= 5;
    // leaf table words per thread: frame-per-unit: LEAF_COUNT leaves x N words (the same for all M
    // words of the thread); group-per-unit: the dead-end leaf only, one copy per word (M x N)
    static constexpr int LEAF_WORDS = FRAME_PER_UNIT ? LEAF_COUNT * N : M * N;
    static constexpr uint32_t LOWER_MODE = LOWER_LEAF_DEAD | (P_LEAF ? LOWER_LEAF_P : 0u);
    static_assert(N >= 1 && N <= 6 && K >= 0 && K <= 4 && DMAX >= 1 && DMAX <= UC_DMAX, "shape");
    static_assert(N * N + KN >= LOW, "too few models for one group");
};

__device__ __forceinline__ constexpr uint32_t lane_pattern(int pos) {
    return pos == 0 ? 0xAAAAAAAAu : pos == 1 ? 0xCCCCCCCCu : pos == 2 ? 0xF0F0F0F0u
         : pos == 3 ? 0xFF00FF00u : 0xFFFF0000u;
}

template <int F> __device__ __forceinline__ uint32_t bool_fn(uint32_t a, uint32_t b) {
    return (F == BF_AND) ? (a & b) : (F == BF_OR) ? (a | b) : (F == BF_ANDN) ? (a & ~b) : (~a & b);
}

template <class C, int TPB>
struct SlicedThread {
    static constexpr int N = C::N, M = C::M;
    static constexpr int DMAX = C::DMAX;
    uint32_t D[DMAX][M][N];           // register stack
    uint32_t E[N * N];                // thread-uniform edge masks (where not constant)
    uint32_t VH[C::PASS_BITS > 0 ? C::PASS_BITS : 1];   // pass-dependent valuation masks
    const uint32_t *leaf;             // this thread's column of the shared-memory leaf table

    // word of the edge w->u for the thread's m-th word
    __device__ __forceinline__ uint32_t edge(int m, int w, int u) const {
        if (C::FRAME_PER_UNIT) return E[w * N + u];
        const int pos = C::KN + w * N + u;
        if (pos < 5) return lane_pattern(pos);
        if (pos < C::LOW) return ((m >> (pos - 5)) & 1) ? 0xFFFFFFFFu : 0u;
        return E[w * N + u];
    }
    // word of "p_i holds at world w" for the thread's m-th word
    __device__ __forceinline__ uint32_t atom(int i, int m, int w) const {
        const int pos = i * N + w;
        if (pos < 5) return lane_pattern(pos);
        if (pos < C::LOW) return ((m >> (pos - 5)) & 1) ? 0xFFFFFFFFu : 0u;
        return VH[(pos - C::LOW) < C::PASS_BITS ? (pos - C::LOW) : 0];
    }
    // leaf-table word (entry l, world w) - frame-per-unit layout; (word m, world w) otherwise
    __device__ __forceinline__ uint32_t leaf_word(uint32_t l, int m, int w) const {
        if (C::FRAME_PER_UNIT) return leaf[(l * N + w) * TPB];
        return leaf[(m * N + w) * TPB];
    }

    // Once per scan unit: the derived leaves go to the leaf table.
    __device__ __forceinline__ void store_leaves(uint32_t *col) const {
        if (C::FRAME_PER_UNIT) {
#pragma unroll
            for (int w = 0; w < N; ++w) {
                uint32_t none = 0xFFFFFFFFu, boxp = 0xFFFFFFFFu, diap = 0u;
#pragma unroll
                for (int u = 0; u < N; ++u) {
                    none &= ~E[w * N + u];                                   // box F: no successor
                    if (C::P_LEAF) {
                        boxp &= (lane_pattern(u) | ~E[w * N + u]);           // box p_0
                        diap |= (lane_pattern(u) & E[w * N + u]);            // dia p_0
                    }
                }
                col[(LEAF_DEAD * N + w) * TPB] = none;
                if (C::P_LEAF) {
                    col[(LEAF_P * N + w) * TPB] = lane_pattern(w);
                    col[(LEAF_BOXP * N + w) * TPB] = boxp;
                    col[(LEAF_DIAP * N + w) * TPB] = diap;
                }
            }
        } else {
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) {
                    uint32_t none = 0xFFFFFFFFu;
#pragma unroll
                    for (int u = 0; u < N; ++u) none &= ~edge(m, w, u);
                    col[(m * N + w) * TPB] = none;
                }
        }
    }

    template <int d> __device__ __forceinline__ void load_var(int i) {
        if (d >= DMAX || i >= C::K || (C::P_LEAF && i == 0)) return;   // never emitted for this instantiation
        constexpr int dd = d < DMAX ? d : 0;
#pragma unroll
        for (int m = 0; m < M; ++m)
#pragma unroll
            for (int w = 0; w < N; ++w) D[dd][m][w] = atom(i, m, w);
    }
    template <int d, int F> __device__ __forceinline__ void bool_var(int i) {
        if (d >= DMAX || i >= C::K || (C::P_LEAF && i == 0)) return;
        constexpr int dd = d < DMAX ? d : 0;
#pragma unroll
        for (int m = 0; m < M; ++m)
#pragma unroll
            for (int w = 0; w < N; ++w) D[dd][m][w] = bool_fn<F>(D[dd][m][w], atom(i, m, w));
    }
    template <int d> __device__ __forceinline__ void load_leaf(uint32_t l) {
        if (d >= DMAX) return;
        constexpr int dd = d < DMAX ? d : 0;
        if (C::FRAME_PER_UNIT) {
            uint32_t v[N];
#pragma unroll
            for (int w = 0; w < N; ++w) v[w] = leaf_word(l, 0, w);
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) D[dd][m][w] = v[w];
        } else {
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) D[dd][m][w] = leaf_word(l, m, w);
        }
    }
    template <int d, int F> __device__ __forceinline__ void bool_leaf(uint32_t l) {
        if (d >= DMAX) return;
        constexpr int dd = d < DMAX ? d : 0;
        if (C::FRAME_PER_UNIT) {
            uint32_t v[N];
#pragma unroll
            for (int w = 0; w < N; ++w) v[w] = leaf_word(l, 0, w);
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) D[dd][m][w] = bool_fn<F>(D[dd][m][w], v[w]);
        } else {
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) D[dd][m][w] = bool_fn<F>(D[dd][m][w], leaf_word(l, m, w));
        }
    }
    template <int d> __device__ __forceinline__ void load_zero() {
        if (d >= DMAX) return;
        constexpr int dd = d < DMAX ? d : 0;
#pragma unroll
        for (int m = 0; m < M; ++m)
#pragma unroll
            for (int w = 0; w < N; ++w) D[dd][m][w] = 0u;
    }
    template <int d> __device__ __forceinline__ void box() {
        if (d >= DMAX) return;
        constexpr int dd = d < DMAX ? d : 0;
#pragma unroll
        for (int m = 0; m < M; ++m) {
            uint32_t r[N];
#pragma unroll
            for (int w = 0; w < N; ++w) {
                uint32_t acc = 0xFFFFFFFFu;
#pragma unroll
                for (int u = 0; u < N; ++u) acc &= (D[dd][m][u] | ~edge(m, w, u));
                r[w] = acc;
            }
#pragma unroll
            for (int w = 0; w < N; ++w) D[dd][m][w] = r[w];
        }
    }
    template <int d> __device__ __forceinline__ void dia() {
        if (d >= DMAX) return;
        constexpr int dd = d < DMAX ? d : 0;
#pragma unroll
        for (int m = 0; m < M; ++m) {
            uint32_t r[N];
#pragma unroll
            for (int w = 0; w < N; ++w) {
                uint32_t acc = 0u;
#pragma unroll
                for (int u = 0; u < N; ++u) acc |= (D[dd][m][u] & edge(m, w, u));
                r[w] = acc;
            }
#pragma unroll
            for (int w = 0; w < N; ++w) D[dd][m][w] = r[w];
        }
    }
    // ---- fused forms (ucode.h, LOWER_FUSE): the operand is read where it lives ----------------------
    // D[0] <- box / dia p_I: the compile-time bits of the atom fold into the logic, and since the
    // source is not D[0] the result needs no staging copy
    template <int I, bool BOX> __device__ __forceinline__ void modal_var0() {
        if (I >= C::K || (C::P_LEAF && I == 0)) return;
#pragma unroll
        for (int m = 0; m < M; ++m)
#pragma unroll
            for (int w = 0; w < N; ++w) {
                uint32_t acc = BOX ? 0xFFFFFFFFu : 0u;
#pragma unroll
                for (int u = 0; u < N; ++u) {
                    if (BOX) acc &= (atom(I, m, u) | ~edge(m, w, u));
                    else acc |= (atom(I, m, u) & edge(m, w, u));
                }
                D[0][m][w] = acc;
            }
    }
    // D[d] <- box / dia leaf; with one frame per thread the leaf and the edge masks are the same for
    // all M words, so the N results are computed once
    template <int d, bool BOX> __device__ __forceinline__ void modal_leaf(uint32_t l) {
        if (d >= DMAX) return;
        constexpr int dd = d < DMAX ? d : 0;
        if (C::FRAME_PER_UNIT) {
            uint32_t v[N], r[N];
#pragma unroll
            for (int u = 0; u < N; ++u) v[u] = leaf_word(l, 0, u);
#pragma unroll
            for (int w = 0; w < N; ++w) {
                uint32_t acc = BOX ? 0xFFFFFFFFu : 0u;
#pragma unroll
                for (int u = 0; u < N; ++u) {
                    if (BOX) acc &= (v[u] | ~edge(0, w, u));
                    else acc |= (v[u] & edge(0, w, u));
                }
                r[w] = acc;
            }
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) D[dd][m][w] = r[w];
        } else {
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) {
                    uint32_t acc = BOX ? 0xFFFFFFFFu : 0u;
#pragma unroll
                    for (int u = 0; u < N; ++u) {
                        if (BOX) acc &= (leaf_word(l, m, u) | ~edge(m, w, u));
                        else acc |= (leaf_word(l, m, u) & edge(m, w, u));
                    }
                    D[dd][m][w] = acc;
                }
        }
    }
    template <int d, int F> __device__ __forceinline__ void boolean() {
        if (d + 1 >= DMAX) return;
        constexpr int dd = d + 1 < DMAX ? d : 0, d1 = d + 1 < DMAX ? d + 1 : 1;
#pragma unroll
        for (int m = 0; m < M; ++m)
#pragma unroll
            for (int w = 0; w < N; ++w) D[dd][m][w] = bool_fn<F>(D[dd][m][w], D[d1][m][w]);
    }
    // FIN, kind = 0 ALL, 1 ANY, 2 XOR, 3 XNOR (ucode.h): r[m] = OR_w (D0[w] ^ [pair] D1[w] ^ pol) with
    // pol = all-ones for ALL / XNOR - one warp-uniform formula, no dispatch.
    __device__ __forceinline__ void fin(uint32_t kind, uint32_t (&r)[M]) const {
        const uint32_t pol = ((kind ^ (kind >> 1)) & 1u) ? 0u : 0xFFFFFFFFu;
        if (DMAX > 1 && kind >= 2u) {
            constexpr int d1 = DMAX > 1 ? 1 : 0;
#pragma unroll
            for (int m = 0; m < M; ++m) {
                uint32_t x = 0u;
#pragma unroll
                for (int w = 0; w < N; ++w) x |= D[0][m][w] ^ D[d1][m][w] ^ pol;
                r[m] = x;
            }
            return;
        }
#pragma unroll
        for (int m = 0; m < M; ++m) {
            uint32_t x = 0u;
#pragma unroll
            for (int w = 0; w < N; ++w) x |= D[0][m][w] ^ pol;
            r[m] = x;
        }
    }

    // Runs one lowered program on the thread's M words; r[m] = models that refute / distinguish.
    __device__ __forceinline__ void run(const uint16_t *__restrict__ uc, uint32_t (&r)[M]) {
        uint32_t pc = 0;
        uint32_t nxt = uc[0];
        uint32_t op;
        for (;;) {
            op = nxt & 0xFFu;
            const uint32_t arg = nxt >> 8;
            if (op >= (uint32_t)UC_FIN_ALL && op <= (uint32_t)UC_FIN_XNOR) break;          // FIN
            nxt = uc[++pc];          // prefetch (the slot's stride leaves an entry after FIN)
#define KRIPKE_CASE4(base, call) \
    case (base) + 0: call(0); break; case (base) + 1: call(1); break; \
    case (base) + 2: call(2); break; case (base) + 3: call(3); break;
            switch (op) {
#define KRIPKE_CASE3(base, call) \
    case (base) + 0: call(0); break; case (base) + 1: call(1); break; \
    case (base) + 2: call(2); break;
#define LV0(d) load_var<d>(0)
#define LV1(d) load_var<d>(1)
#define LV2(d) load_var<d>(2)
#define LV3(d) load_var<d>(3)
                KRIPKE_CASE4(UC_LOADV + 0, LV0) KRIPKE_CASE4(UC_LOADV + 4, LV1)
                KRIPKE_CASE4(UC_LOADV + 8, LV2) KRIPKE_CASE4(UC_LOADV + 12, LV3)
#define BV(f, i) KRIPKE_CASE4(UC_BOOLV + ((f) * 4 + (i)) * 4, BVD_##f##_##i)
#define BVD_0_0(d) bool_var<d, 0>(0)
#define BVD_0_1(d) bool_var<d, 0>(1)
#define BVD_0_2(d) bool_var<d, 0>(2)
#define BVD_0_3(d) bool_var<d, 0>(3)
#define BVD_1_0(d) bool_var<d, 1>(0)
#define BVD_1_1(d) bool_var<d, 1>(1)
#define BVD_1_2(d) bool_var<d, 1>(2)
#define BVD_1_3(d) bool_var<d, 1>(3)
#define BVD_2_0(d) bool_var<d, 2>(0)
#define BVD_2_1(d) bool_var<d, 2>(1)
#define BVD_2_2(d) bool_var<d, 2>(2)
#define BVD_2_3(d) bool_var<d, 2>(3)
#define BVD_3_0(d) bool_var<d, 3>(0)
#define BVD_3_1(d) bool_var<d, 3>(1)
#define BVD_3_2(d) bool_var<d, 3>(2)
#define BVD_3_3(d) bool_var<d, 3>(3)
                BV(0, 0) BV(0, 1) BV(0, 2) BV(0, 3) BV(1, 0) BV(1, 1) BV(1, 2) BV(1, 3)
                BV(2, 0) BV(2, 1) BV(2, 2) BV(2, 3) BV(3, 0) BV(3, 1) BV(3, 2) BV(3, 3)
#define LL(d) load_leaf<d>(arg)
#define BL0(d) bool_leaf<d, 0>(arg)
#define BL1(d) bool_leaf<d, 1>(arg)
#define BL2(d) bool_leaf<d, 2>(arg)
#define BL3(d) bool_leaf<d, 3>(arg)
                KRIPKE_CASE4(UC_LOADL, LL)
                KRIPKE_CASE4(UC_BOOLL + 0, BL0) KRIPKE_CASE4(UC_BOOLL + 4, BL1)
                KRIPKE_CASE4(UC_BOOLL + 8, BL2) KRIPKE_CASE4(UC_BOOLL + 12, BL3)
#define BB0(d) boolean<d, 0>()
#define BB1(d) boolean<d, 1>()
#define BB2(d) boolean<d, 2>()
#define BB3(d) boolean<d, 3>()
                KRIPKE_CASE3(UC_BOOL + 0, BB0) KRIPKE_CASE3(UC_BOOL + 4, BB1)
                KRIPKE_CASE3(UC_BOOL + 8, BB2) KRIPKE_CASE3(UC_BOOL + 12, BB3)
#define BOXD(d) box<d>()
#define DIAD(d) dia<d>()
#define LZ(d) load_zero<d>()
                KRIPKE_CASE4(UC_BOX, BOXD)
                KRIPKE_CASE4(UC_DIA, DIAD)
                KRIPKE_CASE4(UC_LOADZ, LZ)
                case UC_BOXV0 + 0: modal_var0<0, true>(); break;  case UC_BOXV0 + 1: modal_var0<1, true>(); break;
                case UC_BOXV0 + 2: modal_var0<2, true>(); break;  case UC_BOXV0 + 3: modal_var0<3, true>(); break;
                case UC_DIAV0 + 0: modal_var0<0, false>(); break; case UC_DIAV0 + 1: modal_var0<1, false>(); break;
                case UC_DIAV0 + 2: modal_var0<2, false>(); break; case UC_DIAV0 + 3: modal_var0<3, false>(); break;
#define BXL(d) modal_leaf<d, true>(arg)
#define DXL(d) modal_leaf<d, false>(arg)
                KRIPKE_CASE4(UC_BOXL, BXL) KRIPKE_CASE4(UC_DIAL, DXL)
#undef BXL
#undef DXL
#undef LV0
#undef LV1
#undef LV2
#undef LV3
#undef BV
#undef LL
#undef BL0
#undef BL1
#undef BL2
#undef BL3
#undef BB0
#undef BB1
#undef BB2
#undef BB3
#undef BOXD
#undef DIAD
#undef LZ
#undef KRIPKE_CASE4
#undef KRIPKE_CASE3
            default: break;
            }
        }
        fin(op - (uint32_t)UC_FIN_ALL, r);
    }
};

// Number of refuted frames inside one thread's group ("group per unit" regime only).
template <class C>
__device__ __forceinline__ uint32_t frames_in_group(const uint32_t (&r)[C::M]) {
    uint32_t cnt = 0;
    if (C::KN >= 5) {                                  // a frame spans 2^(KN-5) whole words
        constexpr int WPF = 1 << (C::KN >= 5 ? C::KN - 5 : 0);
#pragma unroll
        for (int m0 = 0; m0 < C::M; m0 += WPF) {
            uint32_t any = 0;
#pragma unroll
            for (int j = 0; j < WPF; ++j) any |= r[(m0 + j) < C::M ? (m0 + j) : 0];
            cnt += (any != 0u);
        }
    } else {                                           // 2^(5-KN) frames per word, 2^KN bits each
        constexpr int S = 1 << (C::KN < 5 ? C::KN : 0);
        constexpr uint32_t PICK = S == 1 ? 0xFFFFFFFFu : S == 2 ? 0x55555555u : S == 4 ? 0x11111111u
                                : S == 8 ? 0x01010101u : 0x00010001u;
#pragma unroll
        for (int m = 0; m < C::M; ++m) {
            uint32_t y = r[m];
#pragma unroll
            for (int s = 1; s < S; s <<= 1) y |= y >> s;
            cnt += __popc(y & PICK);
        }
    }
    return cnt;
}

template <class C, int TPB, int MINB>
__global__ void __launch_bounds__(TPB, MINB) scan_sliced_kernel(SlicedParams p) {
    constexpr int N = C::N, M = C::M;
    constexpr int SLICED_THREADS = TPB;
    extern __shared__ __align__(16) unsigned char smem[];
    // [leaf table: LEAF_WORDS x TPB words][models u64 x chunk][frames u32 x chunk][best u32 x chunk][ucode]
    uint32_t *s_leaf = reinterpret_cast<uint32_t *>(smem);
    unsigned long long *s_models = reinterpret_cast<unsigned long long *>(s_leaf + C::LEAF_WORDS * TPB);
    uint32_t *s_frames = reinterpret_cast<uint32_t *>(s_models + p.chunk);
    uint32_t *s_best = s_frames + p.chunk;
    uint16_t *s_ucode = reinterpret_cast<uint16_t *>(s_best + p.chunk);

    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t n_items = p.n_ranges * p.n_chunks;
    const uint64_t units_per_item = (uint64_t)p.tiles_per_item * SLICED_THREADS;
    SlicedThread<C, TPB> T;
    T.leaf = s_leaf + threadIdx.x;

    for (uint32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        // (range, chunk) <- item, rotated by the range so that a block's stride through the items does
        // not keep handing it the same program chunk (chunks differ in cost)
        const uint32_t range_id = item / p.n_chunks;
        const uint32_t chunk_id = (item % p.n_chunks + range_id) % p.n_chunks;
        const uint32_t slot0 = chunk_id * p.chunk;
        const uint32_t nslots = min(p.chunk, p.n_slots - slot0);
        const uint64_t u0 = p.unit_begin + (uint64_t)range_id * units_per_item;
        const uint64_t item_units = min(units_per_item, p.unit_begin + p.unit_count - u0);

        // step H1: stage this item's programs in shared memory; zero the block accumulators
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < nslots; i += SLICED_THREADS) {
            s_models[i] = 0ull; s_frames[i] = 0u; s_best[i] = 0xFFFFFFFFu;
        }
        {
            const uint32_t words = nslots * (p.stride / 2);
            const uint32_t *src = reinterpret_cast<const uint32_t *>(p.ucode + (size_t)slot0 * p.stride);
            uint32_t *dst = reinterpret_cast<uint32_t *>(s_ucode);
            for (uint32_t i = threadIdx.x; i < words; i += SLICED_THREADS) dst[i] = src[i];
        }
        __syncthreads();

        for (uint64_t tile = 0; tile * SLICED_THREADS < item_units; ++tile) {
            const uint64_t warp_rel = tile * SLICED_THREADS + (threadIdx.x & ~31u);
            if (warp_rel >= item_units) continue;              // whole warp past the end
            const uint64_t rel = warp_rel + lane;
            const bool valid = rel < item_units;
            const uint64_t unit = u0 + (valid ? rel : 0);

            // steps H2/H3: the thread-uniform index bits become all-0 / all-1 words
            if (C::FRAME_PER_UNIT) {
                const uint64_t f = class_frame(N, p.cls, p.class_table, unit);
#pragma unroll
                for (int e = 0; e < N * N; ++e) T.E[e] = 0u - (uint32_t)((f >> e) & 1ull);
            } else {
#pragma unroll
                for (int e = 0; e < N * N; ++e) {
                    const int pos = C::KN + e;
                    if (pos >= C::LOW) T.E[e] = 0u - (uint32_t)((unit >> (pos - C::LOW)) & 1ull);
                }
            }
            T.store_leaves(s_leaf + threadIdx.x);              // private column: no barrier needed

            for (uint32_t s = 0; s < nslots; ++s) {
                const uint16_t *uc = s_ucode + s * p.stride;
                uint32_t cnt = 0, fcnt = 0;
#pragma unroll 1
                for (uint32_t pass = 0; pass < (1u << C::PASS_BITS); ++pass) {
#pragma unroll
                    for (int j = 0; j < C::PASS_BITS; ++j) T.VH[j] = 0u - ((pass >> j) & 1u);
                    uint32_t r[M];
                    T.run(uc, r);                               // step H4
#pragma unroll
                    for (int m = 0; m < M; ++m) cnt += __popc(r[m]);              // step H5
                    if (!C::FRAME_PER_UNIT) fcnt += frames_in_group<C>(r);
                }
                if (!valid) { cnt = 0; fcnt = 0; }
                // step H6, warp level
                const uint32_t bal = __ballot_sync(0xFFFFFFFFu, cnt != 0u);
                if (bal) {
                    const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);
                    const uint32_t ftot = C::FRAME_PER_UNIT ? (uint32_t)__popc(bal)
                                                            : __reduce_add_sync(0xFFFFFFFFu, fcnt);
                    if (lane == 0) {
                        atomicAdd(&s_models[s], (unsigned long long)tot);
                        atomicAdd(&s_frames[s], ftot);
                        atomicMin(&s_best[s], (uint32_t)warp_rel + (uint32_t)(__ffs(bal) - 1));
                    }
                }
            }
        }

        // step H6, block level: one global atomic triple per (block, program)
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < nslots; i += SLICED_THREADS) {
            if (s_best[i] != 0xFFFFFFFFu) {
                Accum *a = p.accum + p.slot_record[slot0 + i];
                atomicAdd(&a->models, s_models[i] << p.model_shift);
                atomicAdd(&a->frames, (unsigned long long)s_frames[i]);
                atomicMin(&a->best, (unsigned long long)(u0 + s_best[i]) << C::UNIT_FRAME_BITS);
            }
        }
    }
}

// Host launcher for one instantiation.
template <class C, int TPB, int MINB>
int launch_sliced_inst(const ScanJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    // queried for the current device on every call (host-side, microseconds): nothing is cached per process,
    // so several devices and several host threads can use the library
    int blocks_per_sm = 0, sm_count = 0;
    constexpr int SLICED_THREADS = TPB;
    auto kern = scan_sliced_kernel<C, TPB, MINB>;
    const size_t per_slot = 16 + 2 * (size_t)plan.stride;
    const size_t leaf_bytes = (size_t)C::LEAF_WORDS * TPB * sizeof(uint32_t);
    const size_t slot_budget = 32 * 1024;
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(leaf_bytes + slot_budget + 16));
        if (e != cudaSuccess) return (int)e;
        int b = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, kern, SLICED_THREADS, leaf_bytes + slot_budget + 16);
        if (e != cudaSuccess) return (int)e;
        blocks_per_sm = b > 0 ? b : 1;
    }
    const uint64_t frames_per_unit = 1ull << C::UNIT_FRAME_BITS;
    SlicedParams p;
    p.cls = job.cls;
    p.class_table = job.class_table;
    p.unit_begin = job.frame_begin / frames_per_unit;
    p.unit_count = job.frame_count / frames_per_unit;
    p.ucode = plan.ucode; p.slot_record = plan.slot_record;
    p.n_slots = plan.n_slots; p.stride = plan.stride;
    p.model_shift = plan.model_shift;
    p.accum = job.accum;
    if (p.unit_count == 0 || p.n_slots == 0) return 0;

    const uint32_t grid_full = (uint32_t)(sm_count * blocks_per_sm);
    const uint64_t tiles = (p.unit_count + SLICED_THREADS - 1) / SLICED_THREADS;
    const uint32_t chunk_cap = (uint32_t)std::max<size_t>(1, std::min<size_t>(2048, slot_budget / per_slot));
    // Work items: enough of them to balance the grid, each as large as that allows.
    uint32_t chunk;
    uint64_t tiles_per_item;
    if (tiles >= (uint64_t)grid_full * 8) {
        chunk = std::min(p.n_slots, chunk_cap);
        const uint32_t n_chunks = (p.n_slots + chunk - 1) / chunk;
        tiles_per_item = std::max<uint64_t>(1, std::min<uint64_t>(64, tiles * n_chunks / ((uint64_t)grid_full * 16)));
    } else {
        tiles_per_item = 1;
        uint64_t want_chunks = ((uint64_t)grid_full * 4 + tiles - 1) / tiles;
        chunk = (uint32_t)std::max<uint64_t>(8, (p.n_slots + want_chunks - 1) / want_chunks);
        chunk = std::min(std::min(chunk, chunk_cap), p.n_slots);
    }
    p.chunk = chunk;
    p.n_chunks = (p.n_slots + chunk - 1) / chunk;
    p.tiles_per_item = (uint32_t)tiles_per_item;
    const uint64_t n_ranges = (tiles + tiles_per_item - 1) / tiles_per_item;
    // n_ranges * n_chunks must fit 32 bits: split very long scans into several launches
    const uint64_t max_ranges = (0x7FFFFFFFull / p.n_chunks);
    for (uint64_t r0 = 0; r0 < n_ranges; r0 += max_ranges) {
        SlicedParams q = p;
        const uint64_t nr = std::min<uint64_t>(max_ranges, n_ranges - r0);
        q.unit_begin = p.unit_begin + r0 * tiles_per_item * SLICED_THREADS;
        q.unit_count = std::min<uint64_t>(p.unit_count - r0 * tiles_per_item * SLICED_THREADS,
                                          nr * tiles_per_item * SLICED_THREADS);
        q.n_ranges = (uint32_t)nr;
        const uint64_t items = nr * p.n_chunks;
        const uint32_t grid = (uint32_t)std::min<uint64_t>(items, grid_full);
        const size_t smem = leaf_bytes + (size_t)chunk * per_slot + 16;
        kern<<<grid, SLICED_THREADS, smem, (cudaStream_t)stream>>>(q);
        if (launches) ++*launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return (int)e;
    }
    return 0;
}

}  // namespace kripke
