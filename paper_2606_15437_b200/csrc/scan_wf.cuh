// scan_wf.cuh - the warp-frame kernel: fused corpus scan with warp-uniform frames (steps H1-H6).
//
// Layout.  The models of a class scan are numbered X = (c << k*n) | v, c the class-order frame
// index (K: c = f; T: c = the n*(n-1) off-diagonal edge bits), v the valuation index.  The bits of
// X are dealt out, low to high, as
//     [0,5)        the bit position inside a 32-bit word    -> constant words 0xAAAAAAAA, ...
//     [5,10)       the lane                                  -> per-lane all-0 / all-1 words LM[j]
//     [10,10+MB)   which of the thread's M = 2^MB words      -> compile-time
//     [10+MB, ..)  the warp's scan unit G                    -> warp-uniform, used as CONTROL
// With k*n <= 10 every valuation bit is a word or lane bit, so all higher bits are edge bits: the
// frames a warp looks at in one unit differ only in a few low edge bits, and every other edge is
// known to the whole warp.  Box and diamond (Lemma 1) then stop being data
// arithmetic on edge masks: for a world w whose successor row is warp-uniform,
//     box x at w = AND of x[u] over the successors u of w,   dia x at w = OR of the same,
// is selected by a jump on the row's successor mask and costs ceil((s-1)/2) three-input logic
// instructions for s successors - one per row on average over all frames, against n per row when
// the edges are data (scan_sliced.cuh).  Only rows holding word / lane edge bits pay the dense
// price, and the row holding the MB compile-time bits ("m-row", world W0) is unrolled per word.
//
// Typed values (wf_ucode.h).  The M words of a thread are sibling frames that differ in MB edges
// of row W0 only.  A depth-0 subformula is the same for all of them (type S, n registers), a
// depth-1 subformula differs at world W0 only (type H, n-1+M registers), deeper ones are full (type
// F, M*n registers).  The host lowering types every micro-op, so shared work is done once.
//
// Programs travel in the kernel parameter block (constant bank): the interpreter's fetch, decode
// and branch run on the uniform datapath, a block is one warp, and nothing is staged in shared
// memory.  Work item = (program, range of units): the per-lane counters of an item stay in
// registers over the whole range, then one warp reduction and one global atomic triple per item
// (hierarchical reduction: thread -> warp -> one atomic set per item).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "internal.h"

namespace kripke {

struct WfParams {
    uint64_t unit_begin;            // first scan unit (class-order frame index >> UFB)
    uint64_t unit_count;
    uint32_t units_per_item;
    uint32_t n_progs;
    uint32_t n_ranges;              // work items = n_ranges * n_progs
    uint32_t model_shift;           // models count x 2^model_shift (variables the programs ignore)
    Accum *accum;
    const uint32_t *prog_record;    // device: record index per program
    uint16_t prog_off[WF_MAX_PROGS + 2];
    uint16_t ucode[WF_MAX_UCODE];
};
static_assert(sizeof(WfParams) <= 32764, "kernel parameter block too large");

enum { EC_WORD = 0, EC_LANE = 1, EC_MCONST = 2, EC_UNIFORM = 3, EC_ALWAYS = 4 };

template <int N_, int K_, int MB_, int CLS_>
struct WfCfg {
    static constexpr int N = N_, K = K_, MB = MB_, CLS = CLS_;
    static constexpr int M = 1 << MB, KN = K * N;
    static constexpr int LOW = 10 + MB;                       // model-index bits below the unit index
    static constexpr int NFB = (CLS == KRIPKE_CLASS_K) ? N * N : N * (N - 1);   // class-order index bits
    static constexpr int UFB = LOW - KN;                      // log2 frames per unit
    static constexpr uint32_t FULLROW = (1u << N) - 1u;
    static constexpr bool LANE_VAL = KN > 5;                  // valuation bits spread over the lanes

    // position of the edge w -> u in the model index; -1: always present (T's diagonal)
    __host__ __device__ static constexpr int edge_pos(int w, int u) {
        if (CLS == KRIPKE_CLASS_K) return KN + w * N + u;
        if (u == w) return -1;
        return KN + w * (N - 1) + (u < w ? u : u - 1);
    }
    __host__ __device__ static constexpr int edge_class(int w, int u) {
        const int p = edge_pos(w, u);
        return p < 0 ? EC_ALWAYS : p < 5 ? EC_WORD : p < 10 ? EC_LANE : p < LOW ? EC_MCONST : EC_UNIFORM;
    }
    __host__ __device__ static constexpr bool row_pure(int w) {                   // all edges always-present or uniform
        for (int u = 0; u < N; ++u)
            if (edge_class(w, u) != EC_ALWAYS && edge_class(w, u) != EC_UNIFORM) return false;
        return true;
    }
    __host__ __device__ static constexpr int first_pure_row() {
        int w = N;
        while (w > 0 && row_pure(w - 1)) --w;
        return w;
    }
    static constexpr int PR0 = first_pure_row();
    __host__ __device__ static constexpr int m_row() {
        for (int w = 0; w < N; ++w)
            for (int u = 0; u < N; ++u)
                if (edge_class(w, u) == EC_MCONST) return w;
        return -1;
    }
    static constexpr int W0 = m_row();
    __host__ __device__ static constexpr int count_class(int w, int cls) {
        int c = 0;
        for (int u = 0; u < N; ++u) c += edge_class(w, u) == cls;
        return c;
    }
    __host__ __device__ static constexpr bool shape_ok() {
        if (KN > 10 || (KN > 5 && KN != 10) || NFB + KN < LOW || W0 < 0 || PR0 > N - 1) return false;
        for (int w = 0; w < N; ++w) {
            if (w != W0 && count_class(w, EC_MCONST) != 0) return false;     // one m-row only
            if (w != W0 && w < PR0 && count_class(w, EC_UNIFORM) != 0) return false;
            if (w >= PR0 && !row_pure(w)) return false;
        }
        if (count_class(W0, EC_MCONST) != MB) return false;
        // the m-row's uniform edges are bits 0.. of the unit index, in ascending u
        int bit = 0;
        for (int u = 0; u < N; ++u)
            if (edge_class(W0, u) == EC_UNIFORM && edge_pos(W0, u) - LOW != bit++) return false;
        return true;
    }
    static constexpr int NU0 = count_class(W0 < 0 ? 0 : W0, EC_UNIFORM);     // uniform edges of the m-row
    static_assert(shape_ok(), "shape not supported by the warp-frame kernel");
};

__device__ __forceinline__ constexpr uint32_t wf_pattern(int pos) {
    return pos == 0 ? 0xAAAAAAAAu : pos == 1 ? 0xCCCCCCCCu : pos == 2 ? 0xF0F0F0F0u
         : pos == 3 ? 0xFF00FF00u : 0xFFFF0000u;
}

template <int FN> __device__ __forceinline__ uint32_t wf_bool(uint32_t a, uint32_t b) {
    return (FN == BF_AND) ? (a & b) : (FN == BF_OR) ? (a | b) : (FN == BF_ANDN) ? (a & ~b) : (~a & b);
}

// operand kinds of the Boolean micro-ops
enum { VT_S = 0, VT_H = 1, VT_F = 2, VT_ATOM = 3 };

template <class C>
struct WfThread {
    static constexpr int N = C::N, M = C::M, W0 = C::W0;
    uint32_t S[WF_S_SLOTS][N];
    uint32_t Hs[WF_H_SLOTS][N];      // worlds != W0 (entry W0 unused)
    uint32_t Hm[WF_H_SLOTS][M];      // world W0, per sibling
    uint32_t F[2][M][N];
    uint32_t LM[5];                  // lane bit j as an all-0 / all-1 word
    uint32_t G;                      // unit index: the warp-uniform edge bits

    template <int T, int L> __device__ __forceinline__ uint32_t get(int m, int w) const {
        if (T == VT_S) return S[L][w];
        if (T == VT_H) return (w == W0) ? Hm[L][m] : Hs[L][w];
        return F[L][m][w];
    }
    // word of "atom A holds at world w"; A = 0: false, A = 1 + i: p_i   (step H3)
    template <int A> __device__ __forceinline__ uint32_t atom(int w) const {
        if (A == 0 || A > C::K) return 0u;
        const int pos = (A - 1) * N + w;
        return pos < 5 ? wf_pattern(pos) : LM[(pos >= 5 && pos < 10) ? (pos - 5) : 0];
    }
    // word of a data edge (step H2, the few edge bits that vary inside the warp)
    __device__ __forceinline__ uint32_t edge_word(int w, int u) const {
        const int pos = C::edge_pos(w, u);
        return pos < 5 ? wf_pattern(pos < 0 ? 0 : pos) : LM[(pos >= 5 && pos < 10) ? (pos - 5) : 0];
    }

    // ---- modal operators ----------------------------------------------------------------------
    // successor mask of a pure row (runtime w): every edge of the row is warp-uniform
    __device__ __forceinline__ uint32_t row_mask(int w) const {
        if (C::CLS == KRIPKE_CLASS_K) return (G >> (w * N - C::UFB)) & C::FULLROW;
        const uint32_t r = (G >> (w * (N - 1) - C::UFB)) & ((1u << (N - 1)) - 1u);
        return (r & ((1u << w) - 1u)) | (1u << w) | ((r >> w) << (w + 1));
    }
    // R[m] = AND / OR of the operand over the successor set SUB (compile-time)
    template <int ST, int SL, bool BOX, int SUB, int MR>
    __device__ __forceinline__ void row_set(uint32_t (&R)[M]) const {
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            uint32_t acc = BOX ? 0xFFFFFFFFu : 0u;
#pragma unroll
            for (int u = 0; u < N; ++u)
                if ((SUB >> u) & 1) acc = BOX ? (acc & get<ST, SL>(m, u)) : (acc | get<ST, SL>(m, u));
            R[m] = acc;
        }
    }
    // a row with word / lane / compile-time edges (compile-time W); USUB: its uniform edges present
    template <int ST, int SL, bool BOX, int W, int USUB, int MR>
    __device__ __forceinline__ void row_mixed_case(uint32_t (&R)[M]) const {
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            uint32_t acc = BOX ? 0xFFFFFFFFu : 0u;
            int ub = 0;
#pragma unroll
            for (int u = 0; u < N; ++u) {
                const int cls = C::edge_class(W, u);
                const uint32_t x = get<ST, SL>(m, u);
                if (cls == EC_WORD || cls == EC_LANE) {
                    const uint32_t e = edge_word(W, u);
                    acc = BOX ? (acc & (x | ~e)) : (acc | (x & e));          // Lemma 1, per lane
                } else {
                    bool on = cls == EC_ALWAYS;
                    if (cls == EC_MCONST) on = (m >> (C::edge_pos(W, u) - 10)) & 1;
                    if (cls == EC_UNIFORM) { on = (USUB >> ub) & 1; ++ub; }
                    if (on) acc = BOX ? (acc & x) : (acc | x);
                }
            }
            R[m] = acc;
        }
    }
    template <int ST, int SL, bool BOX, int W, int MR>
    __device__ __forceinline__ void row_mixed(uint32_t (&R)[M]) const {
        constexpr int NU = C::count_class(W, EC_UNIFORM);
        if (NU == 0) { row_mixed_case<ST, SL, BOX, W, 0, MR>(R); return; }
        switch (G & ((1u << NU) - 1u)) {
#define WF_MC(c) case c: if constexpr (c < (1 << NU)) row_mixed_case<ST, SL, BOX, W, (c < (1 << NU) ? c : 0), MR>(R); break;
            WF_MC(0) WF_MC(1) WF_MC(2) WF_MC(3) WF_MC(4) WF_MC(5) WF_MC(6) WF_MC(7)
            WF_MC(8) WF_MC(9) WF_MC(10) WF_MC(11) WF_MC(12) WF_MC(13) WF_MC(14) WF_MC(15)
#undef WF_MC
        default: break;
        }
    }
    // destination row w <- R
    template <int DT, int DL, int W, int MR>
    __device__ __forceinline__ void put_row(const uint32_t (&R)[M]) {
        if (DT == VT_H) {
            if (W == W0) {
#pragma unroll
                for (int m = 0; m < M; ++m) Hm[DL][m] = R[MR == 1 ? 0 : m];
            } else {
                Hs[DL][W] = R[0];
            }
        } else {
#pragma unroll
            for (int m = 0; m < M; ++m) F[DL][m][W] = R[MR == 1 ? 0 : m];
        }
    }
    // DT/DL <- box or dia of ST/SL   (S -> H, H -> F, F -> the other F buffer)
    template <int ST, int SL, int DT, int DL, bool BOX>
    __device__ __forceinline__ void modal() {
        uint32_t R[M];
        // rows with data or compile-time edges: unrolled
#define WF_ROW(w)                                                                     \
        if constexpr ((w) < C::PR0 && (w) < N) {                                            \
            constexpr int W = (w) < N ? (w) : 0;                                      \
            constexpr int MR = (ST == VT_S && W != W0) ? 1 : M;                       \
            row_mixed<ST, SL, BOX, W, MR>(R);                                         \
            put_row<DT, DL, W, MR>(R);                                                \
        }
        WF_ROW(0) WF_ROW(1) WF_ROW(2) WF_ROW(3) WF_ROW(4) WF_ROW(5)
#undef WF_ROW
        // pure rows: jump on the successor mask, then store the row
        constexpr int MR = (ST == VT_S) ? 1 : M;
#pragma unroll 1
        for (int w = C::PR0; w < N; ++w) {
            switch (row_mask(w)) {
#define WF_RS(c) case c: if constexpr (c < (1 << N)) row_set<ST, SL, BOX, (c < (1 << N) ? c : 0), MR>(R); break;
#define WF_RS8(b) WF_RS(b) WF_RS(b + 1) WF_RS(b + 2) WF_RS(b + 3) WF_RS(b + 4) WF_RS(b + 5) WF_RS(b + 6) WF_RS(b + 7)
                WF_RS8(0) WF_RS8(8) WF_RS8(16) WF_RS8(24) WF_RS8(32) WF_RS8(40) WF_RS8(48) WF_RS8(56)
#undef WF_RS8
#undef WF_RS
            default: break;
            }
            switch (w) {
#define WF_PUT(c) case c: if constexpr (c >= C::PR0 && c < N) put_row<DT, DL, (c < N ? c : 0), MR>(R); break;
                WF_PUT(0) WF_PUT(1) WF_PUT(2) WF_PUT(3) WF_PUT(4) WF_PUT(5)
#undef WF_PUT
            default: break;
            }
        }
    }

    // ---- Boolean micro-ops --------------------------------------------------------------------
    template <int OT, int OL> __device__ __forceinline__ uint32_t operand(int m, int w) const {
        if (OT == VT_ATOM) return atom<OL>(w);
        return get<(OT == VT_ATOM ? VT_S : OT), (OT == VT_ATOM ? 0 : OL)>(m, w);
    }
    template <int DT, int DL, int OT, int OL, int FN>
    __device__ __forceinline__ void boolean() {
        if (DT == VT_S) {
#pragma unroll
            for (int w = 0; w < N; ++w) S[DL][w] = wf_bool<FN>(S[DL][w], operand<OT, OL>(0, w));
        } else if (DT == VT_H) {
#pragma unroll
            for (int w = 0; w < N; ++w)
                if (w != W0) Hs[DL][w] = wf_bool<FN>(Hs[DL][w], operand<OT, OL>(0, w));
#pragma unroll
            for (int m = 0; m < M; ++m) Hm[DL][m] = wf_bool<FN>(Hm[DL][m], operand<OT, OL>(m, W0));
        } else {
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int w = 0; w < N; ++w) F[DL][m][w] = wf_bool<FN>(F[DL][m][w], operand<OT, OL>(m, w));
        }
    }
    template <int DT, int DL, int FN> __device__ __forceinline__ void boolean_atom(uint32_t a) {
        switch (a) {
        case 1: boolean<DT, DL, VT_ATOM, 1, FN>(); break;
        case 2: boolean<DT, DL, VT_ATOM, 2, FN>(); break;
        default: boolean<DT, DL, VT_ATOM, 0, FN>(); break;
        }
    }
    template <int D, int A> __device__ __forceinline__ void load_atom_c() {
#pragma unroll
        for (int w = 0; w < N; ++w) S[D][w] = atom<A>(w);
    }
    template <int D> __device__ __forceinline__ void load_atom(uint32_t a) {
        switch (a) {
        case 1: load_atom_c<D, 1>(); break;
        case 2: load_atom_c<D, 2>(); break;
        default: load_atom_c<D, 0>(); break;
        }
    }

    // ---- refutation test + counting (step H5) ---------------------------------------------------
    // frames refuted inside one word, valuation bits of the word folded away
    __device__ __forceinline__ static uint32_t frames_in_word(uint32_t r) {
        if (C::KN >= 5) return r != 0u;
        constexpr int SPAN = 1 << (C::KN < 5 ? C::KN : 0);
        constexpr uint32_t PICK = SPAN == 1 ? 0xFFFFFFFFu : SPAN == 2 ? 0x55555555u : SPAN == 4 ? 0x11111111u
                                : SPAN == 8 ? 0x01010101u : 0x00010001u;
#pragma unroll
        for (int s = 1; s < SPAN; s <<= 1) r |= r >> s;
        return __popc(r & PICK);
    }
    template <int T, int L, int POL>
    __device__ __forceinline__ void fin(uint32_t &cnt, uint32_t &fr) const {
        constexpr int MR = (T == VT_S) ? 1 : M;
        uint32_t r[MR];
        if (T == VT_H) {
            uint32_t sh = POL ? 0u : 0xFFFFFFFFu;
#pragma unroll
            for (int w = 0; w < N; ++w)
                if (w != W0) sh = POL ? (sh | Hs[L][w]) : (sh & Hs[L][w]);
#pragma unroll
            for (int m = 0; m < M; ++m) r[m] = POL ? (sh | Hm[L][m]) : ~(sh & Hm[L][m]);
        } else {
#pragma unroll
            for (int m = 0; m < MR; ++m) {
                uint32_t x = POL ? 0u : 0xFFFFFFFFu;
#pragma unroll
                for (int w = 0; w < N; ++w) x = POL ? (x | get<T, L>(m, w)) : (x & get<T, L>(m, w));
                r[m] = POL ? x : ~x;
            }
        }
        uint32_t c = 0;
#pragma unroll
        for (int m = 0; m < MR; ++m) c += __popc(r[m]);
        cnt = c * (M / MR);
        if (C::LANE_VAL) {
            // a frame's valuations are spread over all lanes: one flag bit per sibling, OR over the warp
            uint32_t z = 0;
#pragma unroll
            for (int m = 0; m < MR; ++m) z |= (r[m] != 0u) ? ((MR == 1) ? ((1u << M) - 1u) : (1u << m)) : 0u;
            fr = __popc(__reduce_or_sync(0xFFFFFFFFu, z));
        } else {
            uint32_t f = 0;
#pragma unroll
            for (int m = 0; m < MR; ++m) f += frames_in_word(r[m]);
            fr = f * (M / MR);
        }
    }

    // Runs one lowered program (typed micro-ops, wf_ucode.h) on the current unit.
    __device__ __forceinline__ void run(const WfParams &p, uint32_t pc, uint32_t &cnt, uint32_t &fr) {
        for (;;) {
            const uint32_t ins = p.ucode[pc++];
            const uint32_t arg = ins >> 8;
            switch (ins & 0xFFu) {
#define WF4(base, X) case (base) + 0: X(0) break; case (base) + 1: X(1) break; case (base) + 2: X(2) break; case (base) + 3: X(3) break;
#define WF3(base, X) case (base) + 0: X(0) break; case (base) + 1: X(1) break; case (base) + 2: X(2) break;
#define WF2(base, X) case (base) + 0: X(0) break; case (base) + 1: X(1) break;
#define X_LOADA(d) load_atom<d>(arg);
                WF4(WF_LOADA, X_LOADA)
#define X_BSA0(d) boolean_atom<VT_S, d, 0>(arg);
#define X_BSA1(d) boolean_atom<VT_S, d, 1>(arg);
#define X_BSA2(d) boolean_atom<VT_S, d, 2>(arg);
#define X_BSA3(d) boolean_atom<VT_S, d, 3>(arg);
                WF4(WF_BSA + 0, X_BSA0) WF4(WF_BSA + 4, X_BSA1) WF4(WF_BSA + 8, X_BSA2) WF4(WF_BSA + 12, X_BSA3)
#define X_BSS0(d) boolean<VT_S, d, VT_S, d + 1, 0>();
#define X_BSS1(d) boolean<VT_S, d, VT_S, d + 1, 1>();
#define X_BSS2(d) boolean<VT_S, d, VT_S, d + 1, 2>();
#define X_BSS3(d) boolean<VT_S, d, VT_S, d + 1, 3>();
                WF3(WF_BSS + 0, X_BSS0) WF3(WF_BSS + 4, X_BSS1) WF3(WF_BSS + 8, X_BSS2) WF3(WF_BSS + 12, X_BSS3)
#define X_S2HB(h) modal<VT_S, 0, VT_H, h, true>();
#define X_S2HD(h) modal<VT_S, 0, VT_H, h, false>();
                WF2(WF_S2H + 0, X_S2HB) WF2(WF_S2H + 2, X_S2HD)
#define X_BHA0(h) boolean_atom<VT_H, h, 0>(arg);
#define X_BHA1(h) boolean_atom<VT_H, h, 1>(arg);
#define X_BHA2(h) boolean_atom<VT_H, h, 2>(arg);
#define X_BHA3(h) boolean_atom<VT_H, h, 3>(arg);
                WF2(WF_BHA + 0, X_BHA0) WF2(WF_BHA + 2, X_BHA1) WF2(WF_BHA + 4, X_BHA2) WF2(WF_BHA + 6, X_BHA3)
#define X_BHS0(h) boolean<VT_H, h, VT_S, 0, 0>();
#define X_BHS1(h) boolean<VT_H, h, VT_S, 0, 1>();
#define X_BHS2(h) boolean<VT_H, h, VT_S, 0, 2>();
#define X_BHS3(h) boolean<VT_H, h, VT_S, 0, 3>();
                WF2(WF_BHS + 0, X_BHS0) WF2(WF_BHS + 2, X_BHS1) WF2(WF_BHS + 4, X_BHS2) WF2(WF_BHS + 6, X_BHS3)
            case WF_BHH + 0: boolean<VT_H, 0, VT_H, 1, 0>(); break;
            case WF_BHH + 1: boolean<VT_H, 0, VT_H, 1, 1>(); break;
            case WF_BHH + 2: boolean<VT_H, 0, VT_H, 1, 2>(); break;
            case WF_BHH + 3: boolean<VT_H, 0, VT_H, 1, 3>(); break;
            case WF_H2F + 0: modal<VT_H, 0, VT_F, 0, true>(); break;
            case WF_H2F + 1: modal<VT_H, 0, VT_F, 1, true>(); break;
            case WF_H2F + 2: modal<VT_H, 0, VT_F, 0, false>(); break;
            case WF_H2F + 3: modal<VT_H, 0, VT_F, 1, false>(); break;
            case WF_MF + 0: modal<VT_F, 0, VT_F, 1, true>(); break;
            case WF_MF + 1: modal<VT_F, 1, VT_F, 0, true>(); break;
            case WF_MF + 2: modal<VT_F, 0, VT_F, 1, false>(); break;
            case WF_MF + 3: modal<VT_F, 1, VT_F, 0, false>(); break;
#define X_BFA0(b) boolean_atom<VT_F, b, 0>(arg);
#define X_BFA1(b) boolean_atom<VT_F, b, 1>(arg);
#define X_BFA2(b) boolean_atom<VT_F, b, 2>(arg);
#define X_BFA3(b) boolean_atom<VT_F, b, 3>(arg);
                WF2(WF_BFA + 0, X_BFA0) WF2(WF_BFA + 2, X_BFA1) WF2(WF_BFA + 4, X_BFA2) WF2(WF_BFA + 6, X_BFA3)
#define X_BFS0(b) boolean<VT_F, b, VT_S, 0, 0>();
#define X_BFS1(b) boolean<VT_F, b, VT_S, 0, 1>();
#define X_BFS2(b) boolean<VT_F, b, VT_S, 0, 2>();
#define X_BFS3(b) boolean<VT_F, b, VT_S, 0, 3>();
                WF2(WF_BFS + 0, X_BFS0) WF2(WF_BFS + 2, X_BFS1) WF2(WF_BFS + 4, X_BFS2) WF2(WF_BFS + 6, X_BFS3)
#define X_BFH0(b) boolean<VT_F, b, VT_H, 0, 0>();
#define X_BFH1(b) boolean<VT_F, b, VT_H, 0, 1>();
#define X_BFH2(b) boolean<VT_F, b, VT_H, 0, 2>();
#define X_BFH3(b) boolean<VT_F, b, VT_H, 0, 3>();
                WF2(WF_BFH + 0, X_BFH0) WF2(WF_BFH + 2, X_BFH1) WF2(WF_BFH + 4, X_BFH2) WF2(WF_BFH + 6, X_BFH3)
            case WF_FIN_S + 0: fin<VT_S, 0, 0>(cnt, fr); return;
            case WF_FIN_S + 1: fin<VT_S, 0, 1>(cnt, fr); return;
            case WF_FIN_H + 0: fin<VT_H, 0, 0>(cnt, fr); return;
            case WF_FIN_H + 1: fin<VT_H, 0, 1>(cnt, fr); return;
            case WF_FIN_F + 0: fin<VT_F, 0, 0>(cnt, fr); return;
            case WF_FIN_F + 1: fin<VT_F, 1, 0>(cnt, fr); return;
            case WF_FIN_F + 2: fin<VT_F, 0, 1>(cnt, fr); return;
            default: fin<VT_F, 1, 1>(cnt, fr); return;       // WF_FIN_F + 3
            }
        }
    }
};

template <class C, int MINB>
__global__ void __launch_bounds__(32, MINB) scan_wf_kernel(const __grid_constant__ WfParams p) {
    const uint32_t lane = threadIdx.x;
    uint32_t lane_mask[5];
#pragma unroll
    for (int j = 0; j < 5; ++j) lane_mask[j] = 0u - ((lane >> j) & 1u);
    const uint64_t n_items = (uint64_t)p.n_ranges * p.n_progs;
    for (uint64_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        // consecutive items are unit ranges of the SAME program: the warps resident on an SM then run
        // the same micro-ops at about the same time and share instruction and constant cache lines
        const uint32_t prog = (uint32_t)(item / p.n_ranges);
        const uint64_t u0 = (item % p.n_ranges) * p.units_per_item;
        const uint32_t nu = (uint32_t)min((uint64_t)p.units_per_item, p.unit_count - u0);
        const uint32_t pc0 = p.prog_off[prog];
        const uint32_t g0 = (uint32_t)(p.unit_begin + u0);
        uint32_t models = 0, frames = 0, first = 0xFFFFFFFFu;
#pragma unroll 1
        for (uint32_t j = 0; j < nu; ++j) {
            // a fresh register file per (program, unit): nothing of the typed registers is carried
            // from one program run to the next (and the compiler is told so)
            WfThread<C> T;
#pragma unroll
            for (int b = 0; b < 5; ++b) T.LM[b] = lane_mask[b];
            T.G = g0 + j;                                  // steps H2/H3: nothing to decode
            uint32_t cnt, fr;
            T.run(p, pc0, cnt, fr);                        // steps H4/H5
            models += cnt;
            frames += fr;
            first = (cnt != 0u) ? min(first, j) : first;
        }
        // step H6: warp reduction, then one atomic triple per (item = program x unit range)
        const uint32_t tm = __reduce_add_sync(0xFFFFFFFFu, models);
        const uint32_t tf = C::LANE_VAL ? frames : __reduce_add_sync(0xFFFFFFFFu, frames);
        const uint32_t fi = __reduce_min_sync(0xFFFFFFFFu, first);
        if (lane == 0 && fi != 0xFFFFFFFFu) {
            Accum *a = p.accum + p.prog_record[prog];
            atomicAdd(&a->models, (unsigned long long)tm << p.model_shift);
            atomicAdd(&a->frames, (unsigned long long)tf);
            atomicMin(&a->best, (unsigned long long)(p.unit_begin + u0 + fi) << C::UFB);
        }
    }
}

}  // namespace kripke
