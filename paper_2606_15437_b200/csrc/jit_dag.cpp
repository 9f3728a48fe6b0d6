// jit_dag.cpp - the batch graph of the compiled scans (jit.h): postfix programs -> one DAG of distinct
// subterms over the connectives {and, box} with complemented edges.  Pure host code, no CUDA.
//
// Rewrites (all exact identities of the semantics of PAPER.md:38-40):
//   not x           = the edge to x, complemented
//   x or y          = not (not x and not y)          x -> y = not (x and not y)
//   dia x           = not box not x                   (Lemma 1: succ & x != 0  <=>  not (succ subset of ~x))
//   box T           = T ;  x and T = x ;  x and F = F ;  x and x = x ;  x and not x = F
//   box x and box y = box (x and y)                   (box distributes over conjunction on every frame)
// Conjunctions are flattened into sets, sorted and folded left to right, so that equal sets give the
// same node whatever the order and bracketing in the formulas.
#include "jit.h"

#include <algorithm>

namespace kripke {

uint32_t Dag::intern(const DagNode &nd) {
    const std::array<uint32_t, 5> key = {(uint32_t)nd.kind, (uint32_t)nd.var, nd.a, nd.b, nd.salt};
    auto it = index_.find(key);
    if (it != index_.end()) return it->second;
    const uint32_t id = (uint32_t)nodes.size();
    nodes.push_back(nd);
    index_.emplace(key, id);
    return id;
}

uint32_t Dag::lit_const(bool v) {
    DagNode nd{DagNode::CONST0, 0, 0, 0, 0, 0};
    return intern(nd) * 2 + (v ? 1u : 0u);
}

uint32_t Dag::lit_var(uint32_t i) {
    DagNode nd{DagNode::VAR, (uint8_t)i, 0, 0, 0, i < var_rank.size() ? var_rank[i] : (uint8_t)0};
    return intern(nd) * 2;
}

// The conjuncts of a literal: a non-complemented conjunction of this owner expands into its operands.
void Dag::conjuncts(uint32_t lit, std::vector<uint32_t> *out) const {
    const DagNode &nd = nodes[lit >> 1];
    if (!(lit & 1u) && nd.kind == DagNode::AND && nd.salt == salt) {
        conjuncts(nd.a, out);
        conjuncts(nd.b, out);
    } else {
        out->push_back(lit);
    }
}

uint32_t Dag::mk_box(uint32_t x) {
    if (nodes[x >> 1].kind == DagNode::CONST0 && (x & 1u)) return x;       // box T = T
    DagNode nd{DagNode::BOX, 0, x, 0, salt, rank_of(x)};
    return intern(nd) * 2;
}

uint32_t Dag::mk_and(uint32_t x, uint32_t y) {
    std::vector<uint32_t> c;
    conjuncts(x, &c);
    conjuncts(y, &c);
    for (;;) {
        std::sort(c.begin(), c.end());
        c.erase(std::unique(c.begin(), c.end()), c.end());
        std::vector<uint32_t> keep, boxed;
        for (size_t i = 0; i < c.size(); ++i) {
            const uint32_t l = c[i];
            const DagNode &nd = nodes[l >> 1];
            if (nd.kind == DagNode::CONST0) {
                if (!(l & 1u)) return lit_const(false);                    // ... and F
                continue;                                                  // ... and T
            }
            if (i + 1 < c.size() && c[i + 1] == (l ^ 1u)) return lit_const(false);   // x and not x
            if (merge_boxes && !(l & 1u) && nd.kind == DagNode::BOX && nd.salt == salt) boxed.push_back(nd.a);
            else keep.push_back(l);
        }
        if (boxed.size() < 2) {
            if (boxed.size() == 1) keep.push_back(mk_box(boxed[0]));
            c.swap(keep);
            break;
        }
        uint32_t inner = boxed[0];                                         // box x and box y = box (x and y)
        for (size_t i = 1; i < boxed.size(); ++i) inner = mk_and(inner, boxed[i]);
        keep.push_back(mk_box(inner));
        c.swap(keep);                                                      // the new box may fold again
    }
    std::sort(c.begin(), c.end());
    c.erase(std::unique(c.begin(), c.end()), c.end());
    if (c.empty()) return lit_const(true);
    // fold order: conjuncts of low loop level first (all ranks are 0 in a canonical graph: literal order)
    std::stable_sort(c.begin(), c.end(), [&](uint32_t p, uint32_t q) { return rank_of(p) < rank_of(q); });
    uint32_t acc = c[0];
    for (size_t i = 1; i < c.size(); ++i) {
        DagNode nd{DagNode::AND, 0, std::min(acc, c[i]), std::max(acc, c[i]), salt, std::max(rank_of(acc), rank_of(c[i]))};
        acc = intern(nd) * 2;
    }
    return acc;
}

uint32_t Dag::build(const uint8_t *code, uint32_t len, const uint8_t *rename, uint32_t neg_mask) {
    std::vector<uint32_t> st;
    for (uint32_t i = 0; i < len; ++i) {
        const uint8_t c = code[i];
        if (c == KRIPKE_OP_TOP) st.push_back(lit_const(true));
        else if (c == KRIPKE_OP_BOT) st.push_back(lit_const(false));
        else if (c >= KRIPKE_OP_VAR0 && c < KRIPKE_OP_VAR0 + KRIPKE_MAX_VARS)
            st.push_back(lit_var(rename ? rename[c - KRIPKE_OP_VAR0] : (uint32_t)(c - KRIPKE_OP_VAR0)) ^
                         ((neg_mask >> (c - KRIPKE_OP_VAR0)) & 1u));
        else if (c == KRIPKE_OP_NOT) st.back() ^= 1u;
        else if (c == KRIPKE_OP_BOX) st.back() = mk_box(st.back());
        else if (c == KRIPKE_OP_DIA) st.back() = mk_box(st.back() ^ 1u) ^ 1u;
        else {
            const uint32_t y = st.back(); st.pop_back();
            const uint32_t x = st.back(); st.pop_back();
            if (c == KRIPKE_OP_AND) st.push_back(mk_and(x, y));
            else if (c == KRIPKE_OP_OR) st.push_back(mk_and(x ^ 1u, y ^ 1u) ^ 1u);
            else st.push_back(mk_and(x, y ^ 1u) ^ 1u);                      // imp
        }
    }
    return st.back();
}

uint32_t Dag::support(uint32_t lit) const {
    const DagNode &nd = nodes[lit >> 1];
    switch (nd.kind) {
    case DagNode::CONST0: return 0;
    case DagNode::VAR: return 1u << nd.var;
    case DagNode::BOX: return support(nd.a);
    default: return support(nd.a) | support(nd.b);
    }
}

uint32_t Dag::eval(uint32_t lit, uint32_t n, const uint32_t *succ, const uint32_t *val) const {
    const uint32_t full = (1u << n) - 1u;
    const DagNode &nd = nodes[lit >> 1];
    uint32_t t = 0;
    switch (nd.kind) {
    case DagNode::CONST0: t = 0; break;
    case DagNode::VAR: t = val[nd.var] & full; break;
    case DagNode::AND: t = eval(nd.a, n, succ, val) & eval(nd.b, n, succ, val); break;
    case DagNode::BOX: {
        const uint32_t x = eval(nd.a, n, succ, val);
        for (uint32_t w = 0; w < n; ++w)
            if ((succ[w] & ~x & full) == 0u) t |= 1u << w;                 // Lemma 1, eq. (1)
        break;
    }
    }
    return (lit & 1u) ? (full & ~t) : t;
}

std::string Dag::text(uint32_t lit) const {
    const DagNode &nd = nodes[lit >> 1];
    std::string s = (lit & 1u) ? "~" : "";
    switch (nd.kind) {
    case DagNode::CONST0: return s + "0";
    case DagNode::VAR: return s + (char)('a' + nd.var);
    case DagNode::BOX: return s + "[" + text(nd.a) + "]";
    default: {
        std::vector<uint32_t> c;
        conjuncts(lit & ~1u, &c);
        std::vector<std::string> parts;
        for (uint32_t l : c) parts.push_back(text(l));
        std::sort(parts.begin(), parts.end());
        s += "(";
        for (size_t i = 0; i < parts.size(); ++i) s += (i ? "&" : "") + parts[i];
        return s + ")";
    }
    }
}

namespace {

// Work a literal's cone does inside the loops: box n*n, conjunction n, for the nodes that mention a loop variable.
// `value`: false while still inside the positive conjunctions and boxes at the top of a single formula, which the
// guarded form never evaluates (jit.h).
void loop_cost(const Dag &d, uint32_t lit, bool value, uint32_t n, uint32_t loop_var_mask, std::vector<char> *seen, uint64_t *cost) {
    const DagNode &nd = d.nodes[lit >> 1];
    if (nd.kind != DagNode::AND && nd.kind != DagNode::BOX) return;
    if (!value && !(lit & 1u)) {
        loop_cost(d, nd.a, false, n, loop_var_mask, seen, cost);
        if (nd.kind == DagNode::AND) loop_cost(d, nd.b, false, n, loop_var_mask, seen, cost);
        return;
    }
    if ((*seen)[lit >> 1]) return;
    (*seen)[lit >> 1] = 1;
    if (d.support(lit) & loop_var_mask) *cost += nd.kind == DagNode::BOX ? n * n : n;
    loop_cost(d, nd.a, true, n, loop_var_mask, seen, cost);
    if (nd.kind == DagNode::AND) loop_cost(d, nd.b, true, n, loop_var_mask, seen, cost);
}

}  // namespace

void canonical_rename(const uint8_t *code_a, uint32_t len_a, const uint8_t *code_b, uint32_t len_b,
                      uint32_t support_mask, uint32_t n, uint32_t loop_var_mask, uint8_t *rename_out, uint32_t *neg_out) {
    uint8_t vars[KRIPKE_MAX_VARS];
    uint32_t g = 0;
    for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v) {
        rename_out[v] = 0;
        if ((support_mask >> v) & 1u) vars[g++] = (uint8_t)v;
    }
    uint8_t perm[KRIPKE_MAX_VARS] = {0, 1, 2, 3};
    std::string best;
    uint64_t best_cost = 0;
    bool have = false;
    if (neg_out) *neg_out = 0;
    do {
      for (uint32_t pol = 0; pol < (neg_out ? 1u << g : 1u); ++pol) {
        uint8_t rn[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
        uint32_t neg = 0;
        for (uint32_t i = 0; i < g; ++i) {
            rn[vars[i]] = perm[i];
            if ((pol >> i) & 1u) neg |= 1u << vars[i];
        }
        Dag d;
        const uint32_t la = d.build(code_a, len_a, rn, neg);
        std::string t = d.text(la);
        uint64_t cost = 0;
        if (code_b) {
            const uint32_t lb = d.build(code_b, len_b, rn, neg);
            const std::string tb = d.text(lb);
            t = (t < tb) ? t + "#" + tb : tb + "#" + t;
            std::vector<char> seen(d.nodes.size(), 0);
            loop_cost(d, la, true, n, loop_var_mask, &seen, &cost);
            loop_cost(d, lb, true, n, loop_var_mask, &seen, &cost);
        } else {
            std::vector<char> seen(d.nodes.size(), 0);
            loop_cost(d, la, false, n, loop_var_mask, &seen, &cost);
        }
        if (!have || cost < best_cost || (cost == best_cost && t < best)) {
            best = t;
            best_cost = cost;
            have = true;
            for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v) rename_out[v] = rn[v];
            if (neg_out) *neg_out = neg;
        }
      }
    } while (std::next_permutation(perm, perm + g));
}

}  // namespace kripke
