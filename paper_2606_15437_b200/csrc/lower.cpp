// lower.cpp - host side of step H1 (program staging): validation of postfix programs and their
// lowering to the bit-sliced kernel's micro-ops (ucode.h).  Pure host code, no CUDA.
#include "internal.h"

#include <algorithm>

namespace kripke {

namespace {

bool is_atom(uint8_t c, uint32_t n_vars) {
    return c == KRIPKE_OP_TOP || c == KRIPKE_OP_BOT || (c >= KRIPKE_OP_VAR0 && c < KRIPKE_OP_VAR0 + n_vars);
}
bool is_unary(uint8_t c) { return c == KRIPKE_OP_NOT || c == KRIPKE_OP_BOX || c == KRIPKE_OP_DIA; }
bool is_binary(uint8_t c) { return c == KRIPKE_OP_AND || c == KRIPKE_OP_OR || c == KRIPKE_OP_IMP; }

// Simplified syntax tree used by the lowering.
enum NodeKind : uint8_t { N_CONST, N_VAR, N_NOT, N_BOX, N_DIA, N_AND, N_OR, N_IMP };
struct Node {
    NodeKind kind;
    uint8_t value;   // N_CONST: 0/1, N_VAR: index
    int a, b;        // children
    int need;        // register-stack slots needed to evaluate this subtree
};

struct Leaf {
    bool is = false;      // the subtree is read as an operand, it never occupies a slot
    bool is_var = false;  // true: variable p_id (LOADV / BOOLV); false: leaf-table entry id (LOADL / BOOLL)
    uint8_t id = 0;
    int pol = 0;          // 1 = the subtree's value is the complement of the leaf
};

struct Lowerer {
    uint32_t mode = 0;               // LOWER_LEAF_* flags
    uint8_t rename[KRIPKE_MAX_VARS] = {0, 1, 2, 3};   // variable index -> index in the reduced valuation
    std::vector<Node> nodes;
    std::vector<uint16_t> out;
    uint32_t n_modal = 0, n_bool = 0;

    int add(NodeKind k, uint8_t v, int a, int b) {
        nodes.push_back(Node{k, v, a, b, 0});
        return (int)nodes.size() - 1;
    }
    bool is_const(int i, int v) const { return nodes[i].kind == N_CONST && nodes[i].value == v; }
    bool is_const(int i) const { return nodes[i].kind == N_CONST; }

    // constant folding while building (results are exact identities of the semantics)
    int mk_not(int x) {
        if (is_const(x)) return add(N_CONST, !nodes[x].value, -1, -1);
        if (nodes[x].kind == N_NOT) return nodes[x].a;
        return add(N_NOT, 0, x, -1);
    }
    int mk_modal(NodeKind k, int x) {
        if (k == N_BOX && is_const(x, 1)) return x;   // box T = T
        if (k == N_DIA && is_const(x, 0)) return x;   // dia F = F
        return add(k, 0, x, -1);                      // box F (dead ends) and dia T stay
    }
    int mk_and(int x, int y) {
        if (is_const(x, 0) || is_const(y, 0)) return add(N_CONST, 0, -1, -1);
        if (is_const(x, 1)) return y;
        if (is_const(y, 1)) return x;
        return add(N_AND, 0, x, y);
    }
    int mk_or(int x, int y) {
        if (is_const(x, 1) || is_const(y, 1)) return add(N_CONST, 1, -1, -1);
        if (is_const(x, 0)) return y;
        if (is_const(y, 0)) return x;
        return add(N_OR, 0, x, y);
    }
    int mk_imp(int x, int y) {
        if (is_const(x, 0) || is_const(y, 1)) return add(N_CONST, 1, -1, -1);
        if (is_const(x, 1)) return y;
        if (is_const(y, 0)) return mk_not(x);
        return add(N_IMP, 0, x, y);
    }

    // Postfix -> folded tree.  The program is already validated.
    int build(const uint8_t *code, uint32_t len) {
        std::vector<int> st;
        for (uint32_t i = 0; i < len; ++i) {
            uint8_t c = code[i];
            if (c == KRIPKE_OP_TOP) st.push_back(add(N_CONST, 1, -1, -1));
            else if (c == KRIPKE_OP_BOT) st.push_back(add(N_CONST, 0, -1, -1));
            else if (c >= KRIPKE_OP_VAR0 && c < KRIPKE_OP_VAR0 + KRIPKE_MAX_VARS)
                st.push_back(add(N_VAR, rename[c - KRIPKE_OP_VAR0], -1, -1));
            else if (is_unary(c)) {
                int x = st.back(); st.pop_back();
                st.push_back(c == KRIPKE_OP_NOT ? mk_not(x) : mk_modal(c == KRIPKE_OP_BOX ? N_BOX : N_DIA, x));
            } else {
                int y = st.back(); st.pop_back();
                int x = st.back(); st.pop_back();
                st.push_back(c == KRIPKE_OP_AND ? mk_and(x, y) : c == KRIPKE_OP_OR ? mk_or(x, y) : mk_imp(x, y));
            }
        }
        return st.back();
    }

    // Variables the folded tree still mentions (bit i = p_i, after renaming).
    uint32_t support(int i) const {
        const Node &nd = nodes[i];
        if (nd.kind == N_VAR) return 1u << nd.value;
        uint32_t s = 0;
        if (nd.a >= 0) s |= support(nd.a);
        if (nd.b >= 0) s |= support(nd.b);
        return s;
    }

    // Is the subtree an atom or a derived leaf of the target kernel?
    Leaf leaf_of(int i) const {
        Leaf lf;
        int pol = 0;
        while (nodes[i].kind == N_NOT) { pol ^= 1; i = nodes[i].a; }
        const Node &nd = nodes[i];
        if (nd.kind == N_VAR) {
            lf.is = true; lf.pol = pol;
            if (nd.value == 0 && (mode & LOWER_LEAF_P)) { lf.is_var = false; lf.id = LEAF_P; }
            else { lf.is_var = true; lf.id = nd.value; }
            return lf;
        }
        if (nd.kind != N_BOX && nd.kind != N_DIA) return lf;
        int j = nd.a, cp = 0;
        while (nodes[j].kind == N_NOT) { cp ^= 1; j = nodes[j].a; }
        const bool box = nd.kind == N_BOX;
        if (nodes[j].kind == N_CONST && (mode & LOWER_LEAF_DEAD)) {
            const int c = nodes[j].value ^ cp;
            // box F = "no successor" ; dia T = ~(box F).  (box T and dia F were folded away.)
            if (box && c == 0) { lf.is = true; lf.id = LEAF_DEAD; lf.pol = pol; }
            else if (!box && c == 1) { lf.is = true; lf.id = LEAF_DEAD; lf.pol = pol ^ 1; }
            return lf;
        }
        if (nodes[j].kind == N_VAR && nodes[j].value == 0 && (mode & LOWER_LEAF_P)) {
            // box ~p = ~dia p ; dia ~p = ~box p
            lf.is = true;
            lf.id = (box != (cp != 0)) ? LEAF_BOXP : LEAF_DIAP;
            lf.pol = pol ^ cp;
            return lf;
        }
        return lf;
    }

    // Register-stack slots needed to leave the subtree's value in a slot; leaves used as operands
    // need none.  The deeper operand of a binary node is evaluated first (Sethi-Ullman).
    int need(int i) {
        if (leaf_of(i).is) return nodes[i].need = 0;
        Node &nd = nodes[i];
        switch (nd.kind) {
        case N_CONST: case N_VAR: nd.need = 1; break;
        case N_NOT: nd.need = need(nd.a); break;
        case N_BOX: case N_DIA: nd.need = std::max(1, need(nd.a)); break;
        default: {
            int l = need(nd.a), r = need(nd.b);
            if (l == 0 && r == 0) nd.need = 1;
            else if (l == 0 || r == 0) nd.need = std::max(l, r);
            else nd.need = (l >= r) ? std::max(l, r + 1) : std::max(r, l + 1);
        }
        }
        return nd.need;
    }

    void op(uint32_t code, uint32_t arg = 0) { out.push_back((uint16_t)(code | (arg << 8))); }

    void load_leaf(const Leaf &lf, int d) {
        if (lf.is_var) op(UC_LOADV + lf.id * 4 + d);
        else op(UC_LOADL + d, lf.id);
    }
    // D[d] <- (D[d] ^ a1) & (leaf ^ a2) up to the returned polarity
    int bool_leaf(const Leaf &lf, int d, int a1, int a2, int flip) {
        const int f = (!a1 && !a2) ? BF_AND : (!a1 && a2) ? BF_ANDN : (a1 && !a2) ? BF_NAND : BF_OR;
        if (lf.is_var) op(UC_BOOLV + (f * 4 + lf.id) * 4 + d);
        else op(UC_BOOLL + f * 4 + d, lf.id);
        ++n_bool;
        return (f == BF_OR) ? !flip : flip;          // ~s1 & ~s2 = ~(s1 | s2)
    }

    // Emits micro-ops leaving the value of node i in slot d; returns its polarity (1 = the slot
    // holds the complement of the value).
    int emit(int i, int d) {
        const Leaf self = leaf_of(i);
        if (self.is) { load_leaf(self, d); return self.pol; }
        const Node nd = nodes[i];
        switch (nd.kind) {
        case N_CONST:
            op(UC_LOADZ + d);
            return nd.value;                      // T is the complement of all-false
        case N_VAR:                               // (always a leaf; kept for completeness)
            op(UC_LOADV + nd.value * 4 + d);
            return 0;
        case N_NOT:
            return !emit(nd.a, d);
        case N_BOX: case N_DIA: {
            int p = emit(nd.a, d);
            // box ~s = ~dia s ; dia ~s = ~box s
            bool box = (nd.kind == N_BOX) != (p != 0);
            op((box ? UC_BOX : UC_DIA) + d);
            ++n_modal;
            return p;
        }
        default: {
            // as a conjunction of literals: and = x & y ; or = ~(~x & ~y) ; imp = ~(x & ~y)
            const int negx = (nd.kind == N_OR), negy = (nd.kind != N_AND), flip = (nd.kind != N_AND);
            const Leaf la = leaf_of(nd.a), lb = leaf_of(nd.b);
            if (lb.is) {                          // y is read as an operand (x may be a leaf too)
                int px = emit(nd.a, d);
                return bool_leaf(lb, d, px ^ negx, lb.pol ^ negy, flip);
            }
            if (la.is) {
                int py = emit(nd.b, d);
                return bool_leaf(la, d, py ^ negy, la.pol ^ negx, flip);
            }
            bool a_first = nodes[nd.a].need >= nodes[nd.b].need;
            int first = a_first ? nd.a : nd.b, second = a_first ? nd.b : nd.a;
            int p1 = emit(first, d), p2 = emit(second, d + 1);
            int px = a_first ? p1 : p2, py = a_first ? p2 : p1;
            int ax = px ^ negx, ay = py ^ negy;
            int a1 = a_first ? ax : ay, a2 = a_first ? ay : ax;   // by slot: d, d+1
            const int f = (!a1 && !a2) ? BF_AND : (!a1 && a2) ? BF_ANDN : (a1 && !a2) ? BF_NAND : BF_OR;
            op(UC_BOOL + f * 4 + d);
            ++n_bool;
            return (f == BF_OR) ? !flip : flip;
        }
        }
    }
};

}  // namespace

int validate_programs(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas, uint32_t n_vars,
                      uint32_t *max_stack_out) {
    if (!offsets || n_vars > KRIPKE_MAX_VARS) return KRIPKE_EINVAL;
    if (n_formulas && !code) return KRIPKE_EINVAL;
    uint32_t deepest = 0;
    bool unsupported = false;
    for (uint32_t b = 0; b < n_formulas; ++b) {
        if (offsets[b + 1] < offsets[b]) return KRIPKE_EINVAL;
        uint32_t len = offsets[b + 1] - offsets[b];
        if (len == 0) return KRIPKE_EPROGRAM;
        if (len > KRIPKE_MAX_PROGRAM_LEN) unsupported = true;
        uint32_t sp = 0, top = 0;
        for (uint32_t i = 0; i < len; ++i) {
            uint8_t c = code[offsets[b] + i];
            if (is_atom(c, n_vars)) ++sp;
            else if (is_unary(c)) { if (sp < 1) return KRIPKE_EPROGRAM; }
            else if (is_binary(c)) { if (sp < 2) return KRIPKE_EPROGRAM; --sp; }
            else return KRIPKE_EPROGRAM;
            top = std::max(top, sp);
        }
        if (sp != 1) return KRIPKE_EPROGRAM;
        deepest = std::max(deepest, top);
    }
    if (max_stack_out) *max_stack_out = deepest;
    if (unsupported || deepest > KRIPKE_MAX_STACK) return KRIPKE_EUNSUPPORTED;
    return KRIPKE_OK;
}

uint32_t program_support(const uint8_t *code, uint32_t len) {
    Lowerer lw;
    return lw.support(lw.build(code, len));
}

// LOWER_FUSE: a load followed by a modal operator on the same slot becomes one fused micro-op.
static void fuse_loads(std::vector<uint16_t> &uc) {
    std::vector<uint16_t> out;
    out.reserve(uc.size());
    for (size_t i = 0; i < uc.size(); ++i) {
        const uint32_t op = uc[i] & 0xFFu, arg = uc[i] >> 8;
        if (i + 1 < uc.size()) {
            const uint32_t op2 = uc[i + 1] & 0xFFu;
            if (op < UC_BOOLV) {                                        // LOADV i, d
                const uint32_t iv = op >> 2, d = op & 3u;
                if (d == 0 && op2 == UC_BOX + d) { out.push_back((uint16_t)(UC_BOXV0 + iv)); ++i; continue; }
                if (d == 0 && op2 == UC_DIA + d) { out.push_back((uint16_t)(UC_DIAV0 + iv)); ++i; continue; }
            } else if (op >= UC_LOADL && op < UC_BOOLL) {               // LOADL leaf, d
                const uint32_t d = op - UC_LOADL;
                if (op2 == UC_BOX + d) { out.push_back((uint16_t)((UC_BOXL + d) | (arg << 8))); ++i; continue; }
                if (op2 == UC_DIA + d) { out.push_back((uint16_t)((UC_DIAL + d) | (arg << 8))); ++i; continue; }
            }
        }
        out.push_back(uc[i]);
    }
    uc.swap(out);
}

bool lower_single(const uint8_t *code, uint32_t len, uint32_t mode, const uint8_t *rename, Lowered *out) {
    Lowerer lw;
    lw.mode = mode;
    if (rename) std::copy(rename, rename + KRIPKE_MAX_VARS, lw.rename);
    int root = lw.build(code, len);
    out->need = std::max(1, lw.need(root));
    if (out->need > UC_DMAX) return false;
    int p = lw.emit(root, 0);
    lw.op(p ? UC_FIN_ANY : UC_FIN_ALL);
    if (mode & LOWER_FUSE) fuse_loads(lw.out);
    out->ucode = std::move(lw.out);
    out->n_modal = lw.n_modal;
    out->n_bool = lw.n_bool;
    return true;
}

bool lower_pair(const uint8_t *code_a, uint32_t len_a, const uint8_t *code_b, uint32_t len_b, uint32_t mode,
                const uint8_t *rename, Lowered *out) {
    Lowerer lw;
    lw.mode = mode;
    if (rename) std::copy(rename, rename + KRIPKE_MAX_VARS, lw.rename);
    int ra = lw.build(code_a, len_a);
    int rb = lw.build(code_b, len_b);
    int na = std::max(1, lw.need(ra)), nb = std::max(1, lw.need(rb));
    // XOR is symmetric: evaluate the deeper formula first (slot 0), the other above it (slot 1)
    if (nb > na) { std::swap(ra, rb); std::swap(na, nb); }
    out->need = std::max(na, nb + 1);
    if (out->need > UC_DMAX) return false;
    int pa = lw.emit(ra, 0);
    int pb = lw.emit(rb, 1);
    lw.op(pa == pb ? UC_FIN_XOR : UC_FIN_XNOR);
    if (mode & LOWER_FUSE) fuse_loads(lw.out);
    out->ucode = std::move(lw.out);
    out->n_modal = lw.n_modal;
    out->n_bool = lw.n_bool;
    return true;
}

}  // namespace kripke
