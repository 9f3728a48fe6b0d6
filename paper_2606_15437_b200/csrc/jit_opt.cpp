// jit_opt.cpp - cost-driven redistribution of box over conjunction in the batch graph (jit.h).
// Pure host code, no CUDA.
//
// On every frame box (x & y) = box x & box y (box holds at w iff the operand holds at every
// successor of w).  The canonical graph (jit_dag.cpp) always keeps the left side, which makes equal formulas
// equal graphs.  For evaluation the cheaper side depends on the batch: box x may be needed by another formula
// anyway, or x may depend only on the variable whose bits lie inside the 32-model word, so that box x is
// computed once per scan unit and not once per word.  jit_optimize() starts from the canonical graph and
// repeatedly applies the single rewrite box (x1 & ... & xk) -> box (S1) & ... & box (Sm) - over all box nodes
// and all partitions {S1..Sm} of their conjuncts - that lowers the cost of the needed nodes most, until no
// rewrite lowers it.  The cost of a node is what the emitter generates for it: n instructions per world of a
// box, one per world of a conjunction, each weighted by the loop level at which that world's value changes.
#include "jit.h"

#include <algorithm>
#include <unordered_map>
#include <unordered_set>

namespace kripke {

namespace {

struct Levels {
    const JitLayout &lay;
    explicit Levels(const JitLayout &l) : lay(l) {}
    std::vector<std::array<int8_t, KRIPKE_MAX_WORLDS>> memo;
    std::vector<char> have;

    // loop level of node id at world w
    const std::array<int8_t, KRIPKE_MAX_WORLDS> &of(const Dag &d, uint32_t id) {
        if (memo.size() < d.nodes.size()) { memo.resize(d.nodes.size()); have.resize(d.nodes.size(), 0); }
        if (have[id]) return memo[id];
        const DagNode &nd = d.nodes[id];
        std::array<int8_t, KRIPKE_MAX_WORLDS> r;
        r.fill(0);
        const uint32_t n = lay.n;
        if (nd.kind == DagNode::VAR) {
            for (uint32_t w = 0; w < n; ++w) r[w] = (int8_t)jit_atom_level(lay, nd.var, w);
        } else if (nd.kind == DagNode::AND) {
            const auto a = of(d, nd.a >> 1), b = of(d, nd.b >> 1);
            for (uint32_t w = 0; w < n; ++w) r[w] = std::max(a[w], b[w]);
        } else if (nd.kind == DagNode::BOX) {
            const auto a = of(d, nd.a >> 1);
            for (uint32_t w = 0; w < n; ++w)
                for (uint32_t u = 0; u < n; ++u) r[w] = std::max<int8_t>(r[w], std::max<int8_t>(a[u], (int8_t)jit_edge_level(lay, w, u)));
        }
        memo[id] = r;
        have[id] = 1;
        return memo[id];
    }
    double cost(const Dag &d, uint32_t id) {
        const DagNode &nd = d.nodes[id];
        if (nd.kind != DagNode::AND && nd.kind != DagNode::BOX) return 0.0;
        const auto &lv = of(d, id);
        double c = 0;
        for (uint32_t w = 0; w < lay.n; ++w) c += (nd.kind == DagNode::BOX ? (double)lay.n : 1.0) * jit_level_weight(lay, lv[w]);
        return c;
    }
    // one conjunction of values at the levels of node id
    double and_cost_at(const Dag &d, uint32_t id) {
        const auto &lv = of(d, id);
        double c = 0;
        for (uint32_t w = 0; w < lay.n; ++w) c += jit_level_weight(lay, lv[w]);
        return c;
    }
};

void children(const DagNode &nd, uint32_t out[2], uint32_t *cnt) {
    *cnt = 0;
    if (nd.kind == DagNode::AND) { out[0] = nd.a >> 1; out[1] = nd.b >> 1; *cnt = 2; }
    else if (nd.kind == DagNode::BOX) { out[0] = nd.a >> 1; *cnt = 1; }
}

// conjuncts of a positive AND literal (flattened)
void conjuncts_of(const Dag &d, uint32_t lit, std::vector<uint32_t> *out) {
    const DagNode &nd = d.nodes[lit >> 1];
    if (!(lit & 1u) && nd.kind == DagNode::AND) { conjuncts_of(d, nd.a, out); conjuncts_of(d, nd.b, out); }
    else out->push_back(lit);
}

// every partition of {0..k-1} into blocks, as block index per element (restricted growth strings)
void partitions(uint32_t k, std::vector<std::vector<uint8_t>> *out) {
    std::vector<uint8_t> a(k, 0), mx(k, 0);
    for (;;) {
        out->push_back(a);
        int i = (int)k - 1;
        while (i > 0 && a[i] == mx[i - 1] + 1) --i;       // mx[i-1] = max of a[0..i-1]
        if (i <= 0) break;
        ++a[i];
        mx[i] = std::max(mx[i - 1], a[i]);
        for (uint32_t j = (uint32_t)i + 1; j < k; ++j) { a[j] = 0; mx[j] = mx[i]; }
    }
}

constexpr uint32_t MAX_CONJUNCTS = 5;      // Bell(5) = 52 partitions per box node

}  // namespace

void jit_optimize(const Dag &in, const JitLayout &lay, std::vector<JitRoot> *roots, Dag *out, JitOptStats *stats) {
    // working graph: a copy of the canonical one that keeps conjunctions of boxes and folds by loop level
    auto fresh = [&]() {
        Dag d;
        d.merge_boxes = false;
        d.salt = 0;
        d.var_rank.resize(KRIPKE_MAX_VARS, 0);
        for (uint32_t v = 0; v < KRIPKE_MAX_VARS && v < lay.g; ++v) {
            int r = 0;
            for (uint32_t w = 0; w < lay.n; ++w) r = std::max(r, jit_atom_level(lay, v, w));
            d.var_rank[v] = (uint8_t)r;
        }
        return d;
    };
    // copy of graph `src` into `dst` with node `sub` (UINT32_MAX: none) replaced by literal-builder `repl`
    struct Copier {
        const Dag &src;
        Dag &dst;
        std::vector<uint32_t> memo;      // node -> literal in dst (UINT32_MAX = not yet)
        uint32_t sub = UINT32_MAX;
        const std::vector<std::vector<uint32_t>> *blocks = nullptr;   // the substitute: conjunction of box (block)
        Copier(const Dag &s, Dag &d) : src(s), dst(d), memo(s.nodes.size(), UINT32_MAX) {}
        uint32_t lit(uint32_t l) { return node(l >> 1) ^ (l & 1u); }
        uint32_t node(uint32_t id) {
            if (memo[id] != UINT32_MAX) return memo[id];
            const DagNode &nd = src.nodes[id];
            uint32_t r;
            if (id == sub) {
                r = dst.lit_const(true);
                for (const auto &blk : *blocks) {
                    uint32_t a = dst.lit_const(true);
                    for (uint32_t l : blk) a = dst.mk_and(a, lit(l));
                    r = dst.mk_and(r, dst.mk_box(a));
                }
            } else if (nd.kind == DagNode::CONST0) r = dst.lit_const(false);
            else if (nd.kind == DagNode::VAR) r = dst.lit_var(nd.var);
            else if (nd.kind == DagNode::AND) r = dst.mk_and(lit(nd.a), lit(nd.b));
            else r = dst.mk_box(lit(nd.a));
            memo[id] = r;
            return r;
        }
    };

    Dag cur = fresh();
    {
        Copier cp(in, cur);
        for (JitRoot &r : *roots) r.map_lits([&](uint32_t l) { return cp.lit(l); });
    }
    JitOptStats st;
    for (uint32_t round = 0;; ++round) {
        Levels lv(lay);
        // needed nodes and their reference counts
        std::vector<uint32_t> ref(cur.nodes.size(), 0), stack;
        std::vector<char> need(cur.nodes.size(), 0);
        auto touch = [&](uint32_t id) { if (!need[id]) { need[id] = 1; stack.push_back(id); } ++ref[id]; };
        for (const JitRoot &r : *roots) r.for_each_lit([&](uint32_t l) { touch(l >> 1); });
        while (!stack.empty()) {
            const uint32_t id = stack.back(); stack.pop_back();
            uint32_t ch[2], cnt;
            children(cur.nodes[id], ch, &cnt);
            for (uint32_t i = 0; i < cnt; ++i) touch(ch[i]);
        }
        const size_t n_before = cur.nodes.size();
        double total = 0;
        for (uint32_t id = 0; id < n_before; ++id) if (need[id]) total += lv.cost(cur, id);
        if (round == 0) st.cost_before = total;
        st.cost_after = total;

        double best_gain = 1e-9;
        uint32_t best_node = UINT32_MAX;
        std::vector<std::vector<uint32_t>> best_blocks;
        for (uint32_t id = 0; id < n_before; ++id) {
            const DagNode nd = cur.nodes[id];
            if (!need[id] || nd.kind != DagNode::BOX || (nd.a & 1u) || cur.nodes[nd.a >> 1].kind != DagNode::AND) continue;
            std::vector<uint32_t> conj;
            conjuncts_of(cur, nd.a, &conj);
            if (conj.size() < 2 || conj.size() > MAX_CONJUNCTS) continue;
            // what removing this box frees: itself and whatever only it kept alive
            std::unordered_map<uint32_t, uint32_t> dec;
            std::unordered_set<uint32_t> freed;
            double freed_cost = lv.cost(cur, id);
            freed.insert(id);
            std::vector<uint32_t> work{nd.a >> 1};
            while (!work.empty()) {
                const uint32_t j = work.back(); work.pop_back();
                if (++dec[j] < ref[j]) continue;
                freed.insert(j);
                freed_cost += lv.cost(cur, j);
                uint32_t ch[2], cnt;
                children(cur.nodes[j], ch, &cnt);
                for (uint32_t i = 0; i < cnt; ++i) work.push_back(ch[i]);
            }
            const double join = lv.and_cost_at(cur, id);
            std::vector<std::vector<uint8_t>> parts;
            partitions((uint32_t)conj.size(), &parts);
            for (const auto &p : parts) {
                const uint32_t m = 1u + *std::max_element(p.begin(), p.end());
                if (m < 2) continue;
                std::vector<std::vector<uint32_t>> blocks(m);
                for (size_t i = 0; i < conj.size(); ++i) blocks[p[i]].push_back(conj[i]);
                // the nodes the right side needs that nothing else keeps alive (speculative nodes stay in `cur` as
                // unreferenced garbage until the next copy)
                std::vector<uint32_t> tops;
                for (const auto &blk : blocks) {
                    uint32_t a = cur.lit_const(true);
                    for (uint32_t l : blk) a = cur.mk_and(a, l);
                    tops.push_back(cur.mk_box(a) >> 1);
                }
                double add = (double)(m - 1) * join;
                std::unordered_set<uint32_t> seen;
                std::vector<uint32_t> w2 = tops;
                while (!w2.empty()) {
                    const uint32_t j = w2.back(); w2.pop_back();
                    const bool alive = j < n_before && need[j] && !freed.count(j);
                    if (alive || !seen.insert(j).second) continue;
                    add += lv.cost(cur, j);
                    uint32_t ch[2], cnt;
                    children(cur.nodes[j], ch, &cnt);
                    for (uint32_t i = 0; i < cnt; ++i) w2.push_back(ch[i]);
                }
                const double gain = freed_cost - add;
                if (gain > best_gain) { best_gain = gain; best_node = id; best_blocks = blocks; }
            }
        }
        if (best_node == UINT32_MAX || round >= 4096) break;
        Dag next = fresh();
        Copier cp(cur, next);
        cp.sub = best_node;
        cp.blocks = &best_blocks;
        for (JitRoot &r : *roots) r.map_lits([&](uint32_t l) { return cp.lit(l); });
        cur = std::move(next);
        ++st.rewrites;
    }
    *out = std::move(cur);
    if (stats) *stats = st;
}

std::vector<double> jit_node_costs(const Dag &dag, const JitLayout &lay) {
    Levels lv(lay);
    std::vector<double> c(dag.nodes.size(), 0.0);
    for (uint32_t id = 0; id < dag.nodes.size(); ++id) c[id] = lv.cost(dag, id);
    return c;
}

// ---- guarded roots (jit.h) -------------------------------------------------------------------------
namespace {

void push_guard(const Dag &d, uint32_t depth, uint32_t lit, std::vector<JitGuarded> *out) {
    const DagNode &nd = d.nodes[lit >> 1];
    if (!(lit & 1u) && nd.kind == DagNode::AND) {
        push_guard(d, depth, nd.a, out);
        push_guard(d, depth, nd.b, out);
    } else if (!(lit & 1u) && nd.kind == DagNode::BOX) {
        push_guard(d, depth + 1, nd.a, out);
    } else if (nd.kind == DagNode::CONST0 && (lit & 1u)) {
        // T holds everywhere: no obligation
    } else {
        out->push_back(JitGuarded{depth, lit});
    }
}

}  // namespace

void jit_guard_roots(const Dag &dag, std::vector<JitRoot> *roots) {
    for (JitRoot &r : *roots) {
        if (r.b != UINT32_MAX || !r.guarded.empty()) continue;
        std::vector<JitGuarded> g;
        push_guard(dag, 0, r.a, &g);
        std::sort(g.begin(), g.end());
        g.erase(std::unique(g.begin(), g.end()), g.end());
        if (g.empty()) continue;                          // the formula is T: the emitter folds the constant root
        if (g.size() == 1 && g[0].depth == 0) continue;   // a bare literal: nothing to push through
        r.guarded = std::move(g);
    }
}

bool jit_root_refuted(const Dag &dag, const JitRoot &root, uint32_t n, const uint32_t *succ, const uint32_t *val) {
    const uint32_t full = (1u << n) - 1u;
    if (root.guarded.empty()) {
        const uint32_t ta = dag.eval(root.a, n, succ, val);
        return root.b == UINT32_MAX ? ta != full : ta != dag.eval(root.b, n, succ, val);
    }
    for (const JitGuarded &g : root.guarded) {
        uint32_t s = full;                                // S_0 = W, S_(d+1) = successors of S_d
        for (uint32_t d = 0; d < g.depth; ++d) {
            uint32_t t = 0;
            for (uint32_t w = 0; w < n; ++w) if ((s >> w) & 1u) t |= succ[w] & full;
            s = t;
        }
        if (s & ~dag.eval(g.lit, n, succ, val) & full) return true;
    }
    return false;
}

}  // namespace kripke
