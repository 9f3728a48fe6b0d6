// jit_emit.cpp - layout selection, program grouping and CUDA C emission of the compiled scans (jit.h).
// Pure host code, no CUDA.  What is emitted is documented at jit_emit_kernel below; the fixed part
// of every kernel (parameters, reduction helpers) is jit_prelude.inc.
#include "jit.h"

#include <algorithm>
#include <array>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <set>

namespace kripke {

namespace {

const char *const kPrelude =
#include "jit_prelude.inc"
    ;

constexpr uint32_t LOOP_BITS = 5;      // words per thread aimed at: 2^5 (amortises the unit set-up and the flush)
constexpr uint32_t MAX_SPLIT = 5;      // threads per frame <= 32: the frame's threads sit in one warp

std::string fmt(const char *f, ...) __attribute__((format(printf, 1, 2)));
std::string fmt(const char *f, ...) {
    char buf[256];
    va_list ap;
    va_start(ap, f);
    vsnprintf(buf, sizeof(buf), f, ap);
    va_end(ap);
    return buf;
}

const char *lane_const(uint32_t pos) {
    static const char *const k[5] = {"0xAAAAAAAAu", "0xCCCCCCCCu", "0xF0F0F0F0u", "0xFF00FF00u", "0xFFFF0000u"};
    return k[pos];
}

// Where the value of bit `pos` of the model index X comes from in a thread, as a C expression that is
// an all-0 / all-1 word (or the in-word lane pattern), and at which loop level it changes:
// 0 = fixed for the unit, 1 = changes with the outer (frame) loop, 2 = changes with the inner (valuation) loop.
struct BitSource {
    const JitLayout &lay;
    std::set<uint32_t> used_inner, used_outer, used_unit;
    explicit BitSource(const JitLayout &l) : lay(l) {}
    int level(uint32_t pos) const {
        if (pos < 5) return 0;
        pos -= 5;
        if (pos < lay.inner) return !lay.nest_first || pos + lay.nest_first >= lay.inner ? 2 : 2 + (int)(lay.inner - lay.nest_first - pos);
        pos -= lay.inner;
        if (pos < lay.lane_bits) return 0;
        pos -= lay.lane_bits;
        return pos < lay.outer ? 1 : 0;
    }
    std::string word(uint32_t pos) {
        if (pos < 5) return lane_const(pos);
        pos -= 5;
        if (pos < lay.inner) { used_inner.insert(pos); return fmt("mi%u", pos); }
        pos -= lay.inner;
        if (pos < lay.lane_bits) { used_unit.insert(pos); return fmt("mu%u", pos); }      // low unit bits = the lane
        pos -= lay.lane_bits;
        if (pos < lay.outer) { used_outer.insert(pos); return fmt("mo%u", pos); }
        pos -= lay.outer;
        used_unit.insert(pos + lay.lane_bits);
        return fmt("mu%u", pos + lay.lane_bits);
    }
};

// ---- expressions and their mapping onto 3-input logic instructions ---------------------------------
// Every value of the loop body (one world of one graph node, or a program's refuted-lane word) is a small
// expression tree over operands (other values, masks, lane patterns).  A value with a single use at the same
// loop level is substituted into its consumer; each remaining tree is then covered with 3-input look-up
// tables (LOP3.LUT) by dynamic programming over its cuts - the fewest instructions a tree allows - and
// emitted as lop3.b32 with the table computed here.  What the kernel executes is therefore known
// statically: one LOP3 per emitted table.
struct Ex {
    enum Op : uint8_t { LEAF, CONST, AND, OR, XOR } op;
    bool neg;           // the value is complemented (CONST: false = all-0, true = all-1)
    int a, b;           // operands of a binary node
    std::string tok;    // LEAF: the operand as a C expression
};

struct Emitter {
    const Dag &dag;
    const JitLayout &lay;
    BitSource bits;
    std::set<uint32_t> used_table;          // table classes: edge positions read from the table entry
    std::vector<char> done;
    std::vector<std::array<int8_t, KRIPKE_MAX_WORLDS>> lvl;   // loop level of every (node, world) value
    uint32_t n_box = 0, n_and = 0;

    std::vector<Ex> pool;
    struct Stmt {
        int level;
        std::string out;        // value name; "" = a program's refuted-lane word r
        int root;
        std::string tail;       // text after the value (programs: the count updates)
        bool inlined = false;
        bool keep = false;      // the value is read by literal text: never substitute it away
    };
    std::vector<Stmt> stmts;
    static constexpr int MAX_LEVELS = 2 + 16;
    std::string body[MAX_LEVELS];
    uint64_t ops[MAX_LEVELS] = {0};
    int deep() const { return lay.nest_first ? 2 + (int)(lay.inner - lay.nest_first) : 2; }   // level of the innermost loop
    uint32_t n_tmp = 0;

    Emitter(const Dag &d, const JitLayout &l) : dag(d), lay(l), bits(l), done(d.nodes.size(), 0), lvl(d.nodes.size()) {
        for (auto &x : lvl) x.fill(-1);
    }

    // ---- expression constructors (constants fold) ----
    int leaf(const std::string &tok, bool neg) { pool.push_back(Ex{Ex::LEAF, neg, -1, -1, tok}); return (int)pool.size() - 1; }
    int constant(bool v) { pool.push_back(Ex{Ex::CONST, v, -1, -1, ""}); return (int)pool.size() - 1; }
    int negate(int x) { pool[x].neg = !pool[x].neg; return x; }
    int bin(Ex::Op op, int x, int y) {
        for (int pass = 0; pass < 2; ++pass) {
            if (pool[x].op == Ex::CONST) {
                const bool v = pool[x].neg;
                if (op == Ex::AND) return v ? y : x;
                if (op == Ex::OR) return v ? x : y;
                return v ? negate(y) : y;                                   // XOR
            }
            std::swap(x, y);
        }
        pool.push_back(Ex{op, false, x, y, ""});
        return (int)pool.size() - 1;
    }

    // position in X of "p_i holds at world w" / of the edge w -> u (-1: constant or table entry)
    int atom_pos(uint32_t i, uint32_t w) const { return (int)(i * lay.n + w); }
    int edge_pos(uint32_t w, uint32_t u) const {
        const uint32_t n = lay.n;
        if (lay.table) return -1;
        if (lay.cls == KRIPKE_CLASS_T) return w == u ? -1 : (int)(lay.kn + w * (n - 1) + (u < w ? u : u - 1));   // reflexive_deposit's compact index
        return (int)(lay.kn + w * n + u);
    }
    // word of the edge w -> u; "" = the edge is always present (class T diagonal)
    std::string edge(uint32_t w, uint32_t u) {
        const uint32_t n = lay.n;
        if (lay.table) { used_table.insert(w * n + u); return fmt("me%u", w * n + u); }
        const int pos = edge_pos(w, u);
        return pos < 0 ? std::string() : bits.word((uint32_t)pos);
    }
    int edge_level(uint32_t w, uint32_t u) const {
        const int pos = edge_pos(w, u);
        return pos < 0 ? 0 : bits.level((uint32_t)pos);
    }
    // loop level of literal l at world w (its node must have been visited)
    int lit_level(uint32_t l, uint32_t w) const {
        const DagNode &nd = dag.nodes[l >> 1];
        if (nd.kind == DagNode::CONST0) return 0;
        if (nd.kind == DagNode::VAR) return bits.level((uint32_t)atom_pos(nd.var, w));
        return lvl[l >> 1][w];
    }
    // literal l at world w as an expression
    int lit(uint32_t l, uint32_t w) {
        const DagNode &nd = dag.nodes[l >> 1];
        const bool neg = l & 1u;
        if (nd.kind == DagNode::CONST0) return constant(neg);
        if (nd.kind == DagNode::VAR) return leaf(bits.word((uint32_t)atom_pos(nd.var, w)), neg);
        return leaf(fmt("t%u_%u", l >> 1, w), neg);
    }
    void node(uint32_t id) {
        if (done[id]) return;
        done[id] = 1;
        const DagNode &nd = dag.nodes[id];
        const uint32_t n = lay.n;
        if (nd.kind == DagNode::AND) {
            node(nd.a >> 1);
            node(nd.b >> 1);
            for (uint32_t w = 0; w < n; ++w) {
                const int L = std::max(lit_level(nd.a, w), lit_level(nd.b, w));
                lvl[id][w] = (int8_t)L;
                stmts.push_back(Stmt{L, fmt("t%u_%u", id, w), bin(Ex::AND, lit(nd.a, w), lit(nd.b, w)), ""});
            }
            ++n_and;
        } else if (nd.kind == DagNode::BOX) {
            node(nd.a >> 1);
            // Lemma 1 on 32 models: R[w] = AND_u ( T[u] | ~E[w][u] )
            for (uint32_t w = 0; w < n; ++w) {
                std::vector<std::pair<int, int>> terms;
                for (uint32_t u = 0; u < n; ++u) {
                    const std::string ew = edge(w, u);
                    const int x = lit(nd.a, u);
                    terms.emplace_back(std::max(lit_level(nd.a, u), edge_level(w, u)),
                                       ew.empty() ? x : bin(Ex::OR, x, leaf(ew, true)));
                }
                int L = 0;
                const int acc = fold_by_level(Ex::AND, terms, &L);
                lvl[id][w] = (int8_t)L;
                stmts.push_back(Stmt{L, fmt("t%u_%u", id, w), acc, ""});
            }
            ++n_box;
        }
    }

    // ---- guard sets of the guarded roots (jit.h): S_d[u] = "world u is reachable in exactly d steps" ----
    // Only class K needs them: T, S4 and S5 frames are reflexive, so every S_d is W.
    std::vector<std::array<int8_t, KRIPKE_MAX_WORLDS>> guard_lvl;       // guard_lvl[d - 1][u]
    int guard(uint32_t d, uint32_t u) {
        if (d == 0 || lay.cls != KRIPKE_CLASS_K) return constant(true);
        const uint32_t n = lay.n;
        while (guard_lvl.size() < d) {
            const uint32_t k = (uint32_t)guard_lvl.size() + 1;          // builds S_k from S_(k-1)
            std::array<int8_t, KRIPKE_MAX_WORLDS> lv;
            lv.fill(0);
            for (uint32_t v = 0; v < n; ++v) {
                int L = 0, acc = constant(false);
                for (uint32_t w = 0; w < n; ++w) {
                    L = std::max(L, std::max(edge_level(w, v), k > 1 ? (int)guard_lvl[k - 2][w] : 0));
                    const int e = leaf(edge(w, v), false);
                    acc = bin(Ex::OR, acc, k > 1 ? bin(Ex::AND, leaf(fmt("s%u_%u", k - 1, w), false), e) : e);
                }
                lv[v] = (int8_t)L;
                stmts.push_back(Stmt{L, fmt("s%u_%u", k, v), acc, ""});
            }
            guard_lvl.push_back(lv);
        }
        return leaf(fmt("s%u_%u", d, u), false);
    }

    // conjuncts of a positive conjunction (flattened)
    void flat_conjuncts(uint32_t l, std::vector<uint32_t> *out) const {
        const DagNode &nd = dag.nodes[l >> 1];
        if (!(l & 1u) && nd.kind == DagNode::AND) { flat_conjuncts(nd.a, out); flat_conjuncts(nd.b, out); }
        else out->push_back(l);
    }
    // Conjunction / disjunction of operands that change at different loop levels: the operands of the lower levels
    // are folded first and become a value of their own at that level, so an inner loop only pays for what
    // changes in it.
    int fold_by_level(Ex::Op op, std::vector<std::pair<int, int>> items, int *level_out) {
        std::stable_sort(items.begin(), items.end(), [](const std::pair<int, int> &x, const std::pair<int, int> &y) { return x.first < y.first; });
        int acc = constant(op == Ex::AND), L = 0;
        for (const auto &it : items) {
            if (it.first > L && pool[acc].op != Ex::CONST && pool[acc].op != Ex::LEAF) {
                const std::string name = fmt("y%u", n_tmp++);
                stmts.push_back(Stmt{L, name, acc, ""});
                acc = leaf(name, false);
            }
            L = std::max(L, it.first);
            acc = bin(op, acc, it.second);
        }
        *level_out = L;
        return acc;
    }
    int and_by_level(std::vector<std::pair<int, int>> items, int *level_out) { return fold_by_level(Ex::AND, std::move(items), level_out); }
    // fail word of one obligation: OR_u ( S_depth[u] & ~lit[u] )
    std::map<std::pair<uint32_t, uint32_t>, std::string> obligation_name;
    std::map<std::pair<uint32_t, uint32_t>, int> obligation_level;
    std::vector<uint32_t> value_uses;       // readers of every node's value other than guarded obligations that fold it themselves
    void count_uses(const std::vector<JitRoot> &roots) {
        value_uses.assign(dag.nodes.size(), 0);
        std::vector<char> seen(dag.nodes.size(), 0);
        std::vector<uint32_t> stack;
        auto visit = [&](uint32_t l) { if (!seen[l >> 1]) { seen[l >> 1] = 1; stack.push_back(l >> 1); } };
        auto ref = [&](uint32_t l) { ++value_uses[l >> 1]; visit(l); };
        for (const JitRoot &r : roots) {
            if (r.guarded.empty()) { r.for_each_lit(ref); continue; }
            for (const JitGuarded &g : r.guarded) {
                const bool folds = g.depth > 0 && lay.cls == KRIPKE_CLASS_K && (g.lit & 1u) && dag.nodes[g.lit >> 1].kind == DagNode::AND;
                if (!folds) { ref(g.lit); continue; }
                std::vector<uint32_t> conj;
                flat_conjuncts(g.lit ^ 1u, &conj);
                for (uint32_t c : conj) ref(c);
            }
        }
        while (!stack.empty()) {
            const DagNode &nd = dag.nodes[stack.back()];
            stack.pop_back();
            if (nd.kind == DagNode::AND) { ref(nd.a); ref(nd.b); }
            else if (nd.kind == DagNode::BOX) ref(nd.a);
        }
    }
    int obligation(const JitGuarded &g) {
        const auto key = std::make_pair(g.depth, g.lit);
        auto it = obligation_name.find(key);
        if (it == obligation_name.end()) {
            const bool guarded = g.depth > 0 && lay.cls == KRIPKE_CLASS_K;
            // ~lit is a conjunction: S & x & y is folded by loop level (the guard and the in-word variable do not
            // change inside the loops)
            std::vector<uint32_t> conj;
            // (only when nothing else reads the conjunction's value)
            if (guarded && (g.lit & 1u) && dag.nodes[g.lit >> 1].kind == DagNode::AND) {
                flat_conjuncts(g.lit ^ 1u, &conj);
                for (uint32_t c : conj) node(c >> 1);
                // where another reader needs the conjunction's value anyway, fold only if at most one conjunct
                // changes in the innermost loop (the fold then costs no more than reading that value)
                if (!value_uses.empty() && value_uses[g.lit >> 1] > 0) {
                    int top = 0, at_top = 0;
                    for (uint32_t c : conj)
                        for (uint32_t u = 0; u < lay.n; ++u) top = std::max(top, lit_level(c, u));
                    for (uint32_t c : conj) {
                        int lc = 0;
                        for (uint32_t u = 0; u < lay.n; ++u) lc = std::max(lc, lit_level(c, u));
                        at_top += lc == top;
                    }
                    if (at_top > 1) conj.clear();
                }
            }
            if (conj.empty()) node(g.lit >> 1);
            int L = 0;
            std::vector<std::pair<int, int>> terms;
            for (uint32_t u = 0; u < lay.n; ++u) {
                int term, lu = 0;
                if (conj.empty()) {
                    term = bin(Ex::AND, guard(g.depth, u), negate(lit(g.lit, u)));
                    lu = lit_level(g.lit, u);
                    if (guarded) lu = std::max(lu, (int)guard_lvl[g.depth - 1][u]);
                } else {
                    std::vector<std::pair<int, int>> items;
                    const int gx = guard(g.depth, u);
                    items.emplace_back((int)guard_lvl[g.depth - 1][u], gx);
                    for (uint32_t c : conj) items.emplace_back(lit_level(c, u), lit(c, u));
                    term = and_by_level(items, &lu);
                }
                terms.emplace_back(lu, term);
            }
            const int acc = fold_by_level(Ex::OR, terms, &L);
            const std::string name = fmt("o%u_%u", g.depth, g.lit);
            stmts.push_back(Stmt{L, name, acc, ""});
            it = obligation_name.emplace(key, name).first;
            obligation_level[key] = L;
        }
        return leaf(it->second, false);
    }

    // ---- single-use substitution ----
    void collect_leaves(int x, std::vector<int> *out) const {
        if (pool[x].op == Ex::LEAF) out->push_back(x);
        else if (pool[x].op != Ex::CONST) { collect_leaves(pool[x].a, out); collect_leaves(pool[x].b, out); }
    }
    void substitute() {
        std::map<std::string, int> producer;
        std::map<std::string, int> uses;
        for (size_t i = 0; i < stmts.size(); ++i)
            if (!stmts[i].out.empty()) producer[stmts[i].out] = (int)i;
        std::vector<std::vector<int>> leaves(stmts.size());
        for (size_t i = 0; i < stmts.size(); ++i) {
            if (stmts[i].root < 0) continue;
            collect_leaves(stmts[i].root, &leaves[i]);
            for (int lf : leaves[i]) ++uses[pool[lf].tok];
        }
        for (size_t i = 0; i < stmts.size(); ++i)
            for (int lf : leaves[i]) {
                auto it = producer.find(pool[lf].tok);
                if (it == producer.end() || uses[pool[lf].tok] != 1) continue;
                Stmt &p = stmts[it->second];
                if (p.keep || p.level != stmts[i].level || pool[p.root].op == Ex::CONST) continue;
                const bool neg = pool[lf].neg;
                pool[lf] = pool[p.root];                  // the producer's tree takes the operand's place
                pool[lf].neg = pool[lf].neg != neg;
                p.inlined = true;
            }
    }

    // ---- covering a tree with 3-input tables ----
    struct Cut { std::vector<std::string> elems; uint32_t cost; };
    std::map<int, uint32_t> best_cost;
    std::map<int, Cut> best_cut;
    std::map<int, std::vector<Cut>> all_cuts;
    static std::string key_of(int x) { return fmt("#%d", x); }
    uint32_t elems_cost(const std::vector<std::string> &e) {
        uint32_t c = 0;
        for (const std::string &k : e) if (k[0] == '#') c += best_cost[std::atoi(k.c_str() + 1)];
        return c;
    }
    // the ways to stand for subtree x inside a table of its parent: as one operand, or through any of its cuts
    std::vector<Cut> options(int x) {
        if (pool[x].op == Ex::LEAF) return {Cut{{pool[x].tok}, 0}};
        cover(x);
        std::vector<Cut> o = all_cuts[x];
        o.push_back(Cut{{key_of(x)}, best_cost[x]});
        return o;
    }
    void cover(int x) {
        if (best_cost.count(x)) return;
        const std::vector<Cut> A = options(pool[x].a), B = options(pool[x].b);
        std::vector<Cut> cuts;
        std::set<std::vector<std::string>> seen;
        for (const Cut &ca : A)
            for (const Cut &cb : B) {
                std::vector<std::string> u = ca.elems;
                for (const std::string &k : cb.elems) if (std::find(u.begin(), u.end(), k) == u.end()) u.push_back(k);
                if (u.size() > 3) continue;
                std::sort(u.begin(), u.end());
                if (!seen.insert(u).second) continue;
                cuts.push_back(Cut{u, elems_cost(u)});
            }
        size_t bi = 0;
        for (size_t i = 1; i < cuts.size(); ++i)
            if (cuts[i].cost < cuts[bi].cost || (cuts[i].cost == cuts[bi].cost && cuts[i].elems.size() < cuts[bi].elems.size())) bi = i;
        best_cost[x] = 1 + cuts[bi].cost;
        best_cut[x] = cuts[bi];
        all_cuts[x] = cuts;
    }
    // truth table of subtree x over the operands named in `in` (bit patterns 0xF0, 0xCC, 0xAA)
    uint32_t table(int x, const std::map<std::string, uint32_t> &in, bool top) const {
        const Ex &e = pool[x];
        if (e.op == Ex::LEAF) return (in.at(e.tok) ^ (e.neg ? 0xFFu : 0u)) & 0xFFu;
        if (!top) {
            auto it = in.find(key_of(x));
            if (it != in.end()) return it->second;        // realised separately: its complement is already applied
        }
        const uint32_t a = table(e.a, in, false), b = table(e.b, in, false);
        const uint32_t v = e.op == Ex::AND ? (a & b) : e.op == Ex::OR ? (a | b) : (a ^ b);
        return (v ^ (e.neg ? 0xFFu : 0u)) & 0xFFu;
    }
    // emits the tables of subtree x into `out`; returns the name holding its value
    std::string realise(int x, const std::string &name, int level, std::string *out) {
        cover(x);
        const Cut &c = best_cut[x];
        std::vector<std::string> names;
        std::map<std::string, uint32_t> in;
        static const uint32_t pat[3] = {0xF0u, 0xCCu, 0xAAu};
        for (size_t i = 0; i < c.elems.size(); ++i) {
            const std::string &k = c.elems[i];
            names.push_back(k[0] == '#' ? realise(std::atoi(k.c_str() + 1), fmt("x%u", n_tmp++), level, out) : k);
            in[k] = pat[i];
        }
        while (names.size() < 3) names.push_back(names[0]);
        const uint32_t lut = table(x, in, true);
        *out += "      unsigned " + name + "; asm(\"lop3.b32 %0, %1, %2, %3, " + fmt("0x%02x", lut) + ";\" : \"=r\"(" + name +
                ") : \"r\"(" + names[0] + "), \"r\"(" + names[1] + "), \"r\"(" + names[2] + "));\n";
        ++ops[level];
        return name;
    }
    void emit_all() {
        substitute();
        for (const Stmt &st : stmts) {
            if (st.inlined) continue;
            std::string &out = body[st.level];
            if (st.root < 0) { out += st.tail; continue; }              // literal text (counts, stores)
            const std::string name = st.out.empty() ? "r" : st.out;
            if (st.out.empty()) out += "      {\n";
            const Ex &e = pool[st.root];
            if (e.op == Ex::CONST) out += "      const unsigned " + name + (e.neg ? " = 0xFFFFFFFFu;\n" : " = 0u;\n");
            else if (e.op == Ex::LEAF) {
                out += "      const unsigned " + name + " = " + (e.neg ? "~" : "") + e.tok + ";\n";
                if (e.neg) ++ops[st.level];
            } else realise(st.root, name, st.level, &out);
            if (st.out.empty()) out += "      " + st.tail + " }\n";
        }
    }
};

}  // namespace

int jit_atom_level(const JitLayout &lay, uint32_t var, uint32_t w) {
    return BitSource(lay).level(var * lay.n + w);
}

int jit_edge_level(const JitLayout &lay, uint32_t w, uint32_t u) {
    const uint32_t n = lay.n;
    if (lay.table) return 0;
    if (lay.cls == KRIPKE_CLASS_T) return w == u ? 0 : BitSource(lay).level(lay.kn + w * (n - 1) + (u < w ? u : u - 1));
    return BitSource(lay).level(lay.kn + w * n + u);
}

double jit_level_weight(const JitLayout &lay, int level) {
    if (level <= 0) return 1.0 / (double)(1u << (lay.inner + lay.outer));
    if (level == 1) return 1.0 / (double)(1u << lay.inner);
    // nested: level 2 = the loop over the nest_first slowest bits (2^nest_first iterations per 2^inner words), every
    // further level doubles
    if (!lay.nest_first) return 1.0;
    const uint32_t bits = std::min<uint32_t>(lay.nest_first + ((uint32_t)level - 2u), lay.inner);
    return (double)(1u << bits) / (double)(1u << lay.inner);
}

bool jit_layout(uint32_t n, uint32_t g, uint32_t cls, JitLayout *out) {
    if (n < 1 || n > KRIPKE_MAX_WORLDS || g > KRIPKE_MAX_VARS || cls > KRIPKE_CLASS_S5) return false;
    JitLayout l;
    l.n = n; l.g = g; l.cls = cls; l.kn = g * n;
    l.table = cls == KRIPKE_CLASS_S4 || cls == KRIPKE_CLASS_S5;
    const uint32_t fb = l.table ? 0u : (cls == KRIPKE_CLASS_T ? n * n - n : n * n);   // frame bits inside X
    if (l.kn >= 5) {
        l.inner = std::min(l.kn - 5, LOOP_BITS);
        l.split = l.kn - 5 - l.inner;
        if (l.split > MAX_SPLIT) { l.inner += l.split - MAX_SPLIT; l.split = MAX_SPLIT; }
        if (l.split == 0 && l.inner < LOOP_BITS) l.outer = std::min(LOOP_BITS - l.inner, fb);
        l.unit_frames_log2 = l.outer;
    } else {
        if (l.table || l.kn + fb < 5) return false;       // lanes would have to hold table frames / too few models
        l.outer = std::min(LOOP_BITS, l.kn + fb - 5);
        l.unit_frames_log2 = 5 - l.kn + l.outer;
    }
    l.nest_first = l.inner >= 2 ? 1u : 0u;      // measured: a first loop over 2 / 3 / 4 bits saves registers but not time
    if (out) *out = l;
    return true;
}

bool jit_density_layout(uint32_t n, uint32_t g, uint32_t cls, JitLayout *out) {
    if (n < 1 || n > KRIPKE_MAX_WORLDS || g > KRIPKE_MAX_VARS || cls > KRIPKE_CLASS_S5) return false;
    JitLayout l;
    l.n = n; l.g = g; l.cls = cls; l.kn = g * n;
    l.table = cls == KRIPKE_CLASS_S4 || cls == KRIPKE_CLASS_S5;
    const uint32_t fb = l.table ? 0u : (cls == KRIPKE_CLASS_T ? n * n - n : n * n);
    if (l.kn >= 5) {
        l.inner = l.kn - 5;                               // one thread = one frame: all its valuation words
        if (l.inner > 12) return false;
    } else if (l.kn == 0) {
        if (l.table || fb < 5) return false;              // one frame per lane
        // a warp's 32 words are consecutive (1,024 frames = 4 KB of one output row): coalesced stores
        if (fb >= 10) { l.lane_bits = 5; l.split = 5; }
        l.outer = std::min(LOOP_BITS, fb - 5 - l.lane_bits);
        l.unit_frames_log2 = 5 + l.outer + l.lane_bits;   // of the split threads together
    } else {
        return false;                                     // a frame is a fraction of a word: scalar kernel
    }
    if (out) *out = l;
    return true;
}

std::vector<std::vector<uint32_t>> jit_partition(const Dag &dag, const std::vector<JitRoot> &roots,
                                                 const JitLayout &lay, uint32_t max_roots) {
    const uint32_t n = lay.n;
    const size_t R = roots.size();
    // cone of every root: its AND / BOX nodes, with the cost model of the emitter (box n*n, and n), and its
    // obligations (guarded roots: one fail word each, n instructions, shared by the records that carry it)
    std::vector<std::vector<uint32_t>> cone(R);
    std::vector<uint64_t> cost(dag.nodes.size(), 0);                 // in 1/1024 of an instruction per word
    {
        const std::vector<double> c = jit_node_costs(dag, lay);
        for (size_t i = 0; i < dag.nodes.size(); ++i) cost[i] = (uint64_t)(c[i] * 1024.0 + 0.5);
    }
    {
        std::map<std::pair<uint32_t, uint32_t>, uint32_t> obligation_id;
        std::vector<uint32_t> stamp(dag.nodes.size(), UINT32_MAX), stack;
        for (size_t r = 0; r < R; ++r) {
            stack.clear();
            roots[r].for_each_lit([&](uint32_t l) { stack.push_back(l >> 1); });
            while (!stack.empty()) {
                const uint32_t id = stack.back(); stack.pop_back();
                if (stamp[id] == r) continue;
                stamp[id] = (uint32_t)r;
                const DagNode &nd = dag.nodes[id];
                if (nd.kind == DagNode::AND) { cone[r].push_back(id); stack.push_back(nd.a >> 1); stack.push_back(nd.b >> 1); }
                else if (nd.kind == DagNode::BOX) { cone[r].push_back(id); stack.push_back(nd.a >> 1); }
            }
            for (const JitGuarded &g : roots[r].guarded) {
                auto it = obligation_id.find(std::make_pair(g.depth, g.lit));
                if (it == obligation_id.end()) {
                    it = obligation_id.emplace(std::make_pair(g.depth, g.lit), (uint32_t)cost.size()).first;
                    cost.push_back((uint64_t)n * 1024u);
                }
                cone[r].push_back(it->second);
            }
        }
    }
    auto total = [&](size_t r) { uint64_t c = 0; for (uint32_t id : cone[r]) c += cost[id]; return c; };
    std::vector<std::vector<uint32_t>> groups;
    std::vector<char> left(R, 1), in_union(cost.size(), 0);
    size_t n_left = R;
    while (n_left) {
        // seed: the most expensive root left; then repeatedly the root that adds the least new work
        size_t seed = R;
        uint64_t seed_cost = 0;
        for (size_t r = 0; r < R; ++r)
            if (left[r] && (seed == R || total(r) > seed_cost)) { seed = r; seed_cost = total(r); }
        std::vector<uint32_t> members, touched;
        auto take = [&](size_t r) {
            left[r] = 0; --n_left;
            members.push_back((uint32_t)r);
            for (uint32_t id : cone[r]) if (!in_union[id]) { in_union[id] = 1; touched.push_back(id); }
        };
        take(seed);
        while (members.size() < max_roots && n_left) {
            size_t best = R;
            uint64_t best_add = 0;
            for (size_t r = 0; r < R; ++r) {
                if (!left[r]) continue;
                uint64_t add = 0;
                for (uint32_t id : cone[r]) if (!in_union[id]) add += cost[id];
                if (best == R || add < best_add) { best = r; best_add = add; if (add == 0) break; }
            }
            take(best);
        }
        for (uint32_t id : touched) in_union[id] = 0;
        groups.push_back(std::move(members));
    }
    return groups;
}

// The emitted kernel.  A thread owns one scan unit u: the models X = (u << (5+inner+outer)) | (jo << (5+inner))
// | (ji << 5) | lane.  Every bit of X is one atom bit "p_i at world w" or one edge bit "w -> u" (class K:
// frame index bits; class T: the off-diagonal bits, the diagonal is constant; S4 / S5: the table entry), so
// each becomes a word: the lane pattern (bits 0..4), a loop mask (mi*, mo*) or a unit mask (mu*, me*) -
// steps H2 / H3 without any memory traffic.  The loop body evaluates the group's graph in topological
// order on named registers (step H4) and, per program, the refuted-lane word r, c += popc(r) (step H5).
// After the loops kj_flush reduces per warp and block (step H6).
// Failure-density kernel (D_ij = the fraction of valuation-world pairs on which formula i fails on frame j,
// here as the integer count).  Same graph evaluation; per program the failing-world words g_w = ~T_w are either
// popcounted into the thread's frame count (a thread owns one frame and all its valuation words) or - no
// variables, one frame per lane - added up bit-sliced into three planes, from which the thread writes its 32
// consecutive frames' counts with 16-byte stores.
static std::string emit_density_kernel(const Dag &dag, const JitLayout &lay, const std::vector<JitRoot> &roots,
                                       uint32_t threads, uint32_t min_blocks, JitEmitStats *stats) {
    Emitter em(dag, lay);
    const uint32_t n = lay.n, G = (uint32_t)roots.size();
    const bool lanes_are_frames = lay.kn == 0;
    for (uint32_t r = 0; r < G; ++r) {
        em.node(roots[r].a >> 1);
        std::vector<std::string> g(n);
        for (uint32_t w = 0; w < n; ++w) {
            g[w] = fmt("g%u_%u", r, w);
            Emitter::Stmt st{em.lit_level(roots[r].a, w), g[w], em.negate(em.lit(roots[r].a, w)), ""};
            st.keep = true;
            em.stmts.push_back(st);
        }
        if (!lanes_are_frames) {
            std::string t = fmt("      d%u += ", r);
            for (uint32_t w = 0; w < n; ++w) t += (w ? " + " : "") + ("__popc(" + g[w] + ")");
            em.stmts.push_back(Emitter::Stmt{2, "", -1, t + ";\n"});
        } else {
            // bit-sliced sum of the n failing-world words: planes[i] = bit i of the per-lane count
            std::vector<std::vector<std::string>> col(4);
            col[0] = g;
            uint32_t tmp = 0;
            std::string plane[3] = {"0u", "0u", "0u"};
            for (uint32_t i = 0; i < 3; ++i) {
                while (col[i].size() > 1) {
                    const bool three = col[i].size() >= 3;
                    const std::string a = col[i][0], b = col[i][1], c = three ? col[i][2] : "";
                    col[i].erase(col[i].begin(), col[i].begin() + (three ? 3 : 2));
                    const std::string sum = fmt("h%u_%u", r, tmp++), car = fmt("h%u_%u", r, tmp++);
                    int xs = em.bin(Ex::XOR, em.leaf(a, false), em.leaf(b, false));
                    int cy = em.bin(Ex::AND, em.leaf(a, false), em.leaf(b, false));
                    if (three) {
                        cy = em.bin(Ex::OR, cy, em.bin(Ex::AND, em.leaf(c, false), em.bin(Ex::XOR, em.leaf(a, false), em.leaf(b, false))));
                        xs = em.bin(Ex::XOR, xs, em.leaf(c, false));
                    }
                    Emitter::Stmt s1{2, sum, xs, ""}, s2{2, car, cy, ""};
                    s1.keep = s2.keep = true;
                    em.stmts.push_back(s1);
                    em.stmts.push_back(s2);
                    col[i].push_back(sum);
                    col[i + 1].push_back(car);
                }
                if (col[i].size() == 1) plane[i] = col[i][0];
            }
            std::string t;
            if (lay.lane_bits == 5) {
                // The count of frame l as a 4-bit field at bit l (mod 32) of word z[l % 4]: plane 0 where it is,
                // planes 1 and 2 rotated up by one and two.  The thread's 32 counts go to the warp's staging
                // rows (16-byte chunks, XOR-swizzled: conflict-free both ways), and come back transposed so
                // that every store instruction of the warp writes 512 consecutive bytes of the output row.
                t += "      {\n";
                t += "        const unsigned q1 = __funnelshift_l(" + plane[1] + ", " + plane[1] + ", 1), q2 = __funnelshift_l(" +
                     plane[2] + ", " + plane[2] + ", 2);\n";
                for (uint32_t m = 0; m < 4; ++m) {
                    const uint32_t a0 = 0x11111111u << m, a1 = (a0 << 1) | (a0 >> 31), a2 = (a0 << 2) | (a0 >> 30);
                    t += fmt("        const unsigned z%u = (", m) + plane[0] + fmt(" & 0x%08xu) | (q1 & 0x%08xu) | (q2 & 0x%08xu);\n", a0, a1, a2);
                }
                t += "        __syncwarp();\n";
                for (uint32_t c = 0; c < 8; ++c) {
                    t += fmt("        st_w[%uu ^ sw] = make_uint4(", c);
                    for (uint32_t i = 0; i < 4; ++i) {
                        const uint32_t l = 4 * c + i;
                        t += (i ? ", " : "") + (l ? fmt("__funnelshift_r(z%u, z%u, %u) & 7u", l % 4, l % 4, l) : std::string("z0 & 7u"));
                    }
                    t += ");\n";
                }
                t += "        __syncwarp();\n";
                t += fmt("        if (valid) for (unsigned row = p.row_begin[%u]; row < p.row_begin[%u]; ++row) {\n", r, r + 1);
                t += fmt("          uint4 *o = reinterpret_cast<uint4 *>(p.density + (unsigned long long)p.rows[row] * p.total_frames + "
                         "(((((unit >> 5) << %u) + jo) << 10) - p.frame_base)) + lane;\n", lay.outer);
                for (uint32_t q = 0; q < 8; ++q) {
                    t += fmt("          { uint4 v = ld_w[%uu ^ lw%u]; v.x <<= p.model_shift; v.y <<= p.model_shift; v.z <<= p.model_shift; "
                             "v.w <<= p.model_shift; __stcs(o + %u, v); }\n", 32 * q, q & 1u, 32 * q);
                }
                t += "        }\n      }\n";
            } else {
                t += fmt("      if (valid) for (unsigned row = p.row_begin[%u]; row < p.row_begin[%u]; ++row) {\n", r, r + 1);
                t += fmt("        unsigned *o = p.density + (unsigned long long)p.rows[row] * p.total_frames + ((((unit << %u) + jo) << 5) - p.frame_base);\n", lay.outer);
                for (uint32_t q = 0; q < 8; ++q) {
                    t += fmt("        *reinterpret_cast<uint4 *>(o + %u) = make_uint4(", 4 * q);
                    for (uint32_t i = 0; i < 4; ++i)
                        t += (i ? ", " : "") + ("KJ_CNT3(" + plane[0] + ", " + plane[1] + ", " + plane[2] + fmt(", %u) << p.model_shift", 4 * q + i));
                    t += ");\n";
                }
                t += "      }\n";
            }
            em.stmts.push_back(Emitter::Stmt{2, "", -1, t});
        }
    }
    em.emit_all();

    std::string s = kPrelude;
    s += fmt("\n// density layout: n=%u g=%u cls=%u inner=%u outer=%u unit_frames_log2=%u programs=%u\n", n, lay.g, lay.cls,
             lay.inner, lay.outer, lay.unit_frames_log2, G);
    s += fmt("extern \"C\" __global__ void __launch_bounds__(%u, %u) kripke_jit_scan(const KjParams p) {\n", threads, min_blocks);
    s += "  const unsigned lane = threadIdx.x & 31u;\n";
    if (lay.lane_bits == 5) {
        // staging rows of the warp: thread t owns chunks 8t..8t+7 (its 32 counts); store step q reads chunk (lane & 7) of
        // row 4q + (lane >> 3).  Chunk c of row t lives at 8t + (c ^ (t & 7)).
        s += fmt("  __shared__ uint4 s_stage[%u];\n", threads * 8);
        s += "  uint4 *const st_w = s_stage + (threadIdx.x & ~31u) * 8u + lane * 8u;\n";
        s += "  const unsigned sw = lane & 7u;\n";
        s += "  const uint4 *const ld_w = s_stage + (threadIdx.x & ~31u) * 8u + (lane >> 3) * 8u;\n";
        s += "  const unsigned lw0 = (lane & 7u) ^ (lane >> 3), lw1 = (lane & 7u) ^ (4u + (lane >> 3));\n";
    }
    s += "  for (unsigned item = blockIdx.x; item < p.n_items; item += gridDim.x) {\n";
    s += "    const unsigned long long u0 = p.unit_begin + (unsigned long long)item * p.units_per_item;\n";
    s += "    const unsigned long long rem = p.unit_begin + p.unit_count - u0;\n";
    s += "    const unsigned item_units = rem < p.units_per_item ? (unsigned)rem : p.units_per_item;\n";
    s += fmt("    for (unsigned t0 = 0; t0 < item_units; t0 += %uu) {\n", threads);
    s += "      const unsigned rel = t0 + threadIdx.x;\n";
    s += "      const bool valid = rel < item_units;\n";
    s += "      const unsigned long long unit = u0 + (valid ? rel : 0u);\n";
    s += "      (void)lane;\n";
    for (uint32_t b : em.bits.used_unit) s += fmt("      const unsigned mu%u = 0u - (unsigned)((unit >> %u) & 1ull);\n", b, b);
    if (lay.table) {
        s += "      const unsigned long long frame = p.class_table[unit];\n";
        for (uint32_t e : em.used_table) s += fmt("      const unsigned me%u = 0u - (unsigned)((frame >> %u) & 1ull);\n", e, e);
    }
    s += em.body[0];
    if (!lanes_are_frames) for (uint32_t r = 0; r < G; ++r) s += fmt("      unsigned d%u = 0u;\n", r);
    s += "#pragma unroll 1\n";
    s += fmt("      for (unsigned jo = 0; jo < %uu; ++jo) {\n", 1u << lay.outer);
    for (uint32_t b : em.bits.used_outer) s += fmt("      const unsigned mo%u = 0u - ((jo >> %u) & 1u);\n", b, b);
    s += em.body[1];
    s += "#pragma unroll 1\n";
    s += fmt("      for (unsigned ji = 0; ji < %uu; ++ji) {\n", 1u << lay.inner);
    for (uint32_t b : em.bits.used_inner) s += fmt("      const unsigned mi%u = 0u - ((ji >> %u) & 1u);\n", b, b);
    s += em.body[2];
    s += "      }\n      }\n";
    if (!lanes_are_frames) {
        s += "      if (valid) {\n";
        for (uint32_t r = 0; r < G; ++r)
            s += fmt("        for (unsigned row = p.row_begin[%u]; row < p.row_begin[%u]; ++row) "
                     "p.density[(unsigned long long)p.rows[row] * p.total_frames + (unit - p.frame_base)] = d%u << p.model_shift;\n", r, r + 1, r);
        s += "      }\n";
    }
    s += "    }\n  }\n}\n";
    if (stats) {
        const uint64_t *ops = em.ops;
        stats->logic_ops_emitted = ops[0] + ops[1] + ops[2];
        stats->logic_ops_per_word = (double)ops[2] + (double)ops[1] / (double)(1u << lay.inner) +
                                    (double)ops[0] / (double)(1u << (lay.inner + lay.outer));
        stats->n_box = em.n_box;
        stats->n_and = em.n_and;
    }
    return s;
}

std::string jit_emit_kernel(const Dag &dag, const JitLayout &lay, const std::vector<JitRoot> &roots,
                            uint32_t threads, uint32_t min_blocks, uint32_t mode, JitEmitStats *stats) {
    if (mode == JIT_MODE_DENSITY) return emit_density_kernel(dag, lay, roots, threads, min_blocks, stats);
    Emitter em(dag, lay);
    const uint32_t n = lay.n, G = (uint32_t)roots.size();
    // how refuted FRAMES are counted
    enum { F_MODELS, F_THREAD, F_WORD, F_ANY, F_FOLD } fmode;
    if (lay.kn == 0) fmode = F_MODELS;                              // one valuation: frames = models
    else if (lay.unit_frames_log2 == 0) fmode = F_THREAD;           // the unit lies inside one frame
    else if (lay.kn < 5) fmode = F_FOLD;                            // several frames per word
    else if (lay.inner == 0) fmode = F_WORD;                        // one word per frame
    else fmode = F_ANY;                                             // 2^inner words per frame, several frames per unit
    const bool has_f = fmode == F_WORD || fmode == F_ANY || fmode == F_FOLD;
    const bool packed = lay.inner + lay.outer <= 10;                // models of a unit < 2^16

    em.count_uses(roots);
    for (uint32_t r = 0; r < G; ++r) {
        int e;
        if (!roots[r].guarded.empty()) {
            // refuted lanes of a guarded root: some obligation fails at a world of its guard set (jit.h)
            // Every obligation's fail word is a value of its own: shared by the records of the kernel that carry the
            // same obligation, and computed once per unit when its literal does not change inside the loops.
            std::vector<std::pair<int, int>> items;
            for (const JitGuarded &g : roots[r].guarded) {
                const int x = em.obligation(g);
                items.emplace_back(em.obligation_level[std::make_pair(g.depth, g.lit)], x);
            }
            int L = 0;
            e = em.fold_by_level(Ex::OR, items, &L);
        } else if (roots[r].b == UINT32_MAX) {
            em.node(roots[r].a >> 1);
            // refuted lanes: the truth set is not all worlds
            std::vector<std::pair<int, int>> items;
            for (uint32_t w = 0; w < n; ++w) items.emplace_back(em.lit_level(roots[r].a, w), em.lit(roots[r].a, w));
            int L = 0;
            e = em.negate(em.fold_by_level(Ex::AND, items, &L));
        } else {
            // distinguishing lanes: the two truth sets differ
            em.node(roots[r].a >> 1);
            em.node(roots[r].b >> 1);
            std::vector<std::pair<int, int>> items;
            for (uint32_t w = 0; w < n; ++w)
                items.emplace_back(std::max(em.lit_level(roots[r].a, w), em.lit_level(roots[r].b, w)),
                                   em.bin(Ex::XOR, em.lit(roots[r].a, w), em.lit(roots[r].b, w)));
            int L = 0;
            e = em.fold_by_level(Ex::OR, items, &L);
        }
        // Counters of a unit are 16-bit fields where they fit (a unit has 2^(5+inner+outer) models): with a frame
        // count, models in the low half and frames in the high half of one register; without, two programs per
        // register - half the registers the counters would take.
        std::string tail;
        if (!packed) {
            tail = fmt("c%u += __popc(r);", r);
            if (fmode == F_WORD) tail += fmt(" f%u += (r != 0u);", r);
            else if (fmode == F_ANY) tail += fmt(" a%u |= r;", r);
            else if (fmode == F_FOLD) tail += fmt(" f%u += kj_frames_in_word<%u>(r);", r, lay.kn);
        } else if (has_f) {
            tail = fmt("c%u += __popc(r);", r);
            if (fmode == F_WORD) tail += fmt(" if (r != 0u) c%u += 65536u;", r);
            else if (fmode == F_ANY) tail += fmt(" a%u |= r;", r);
            else tail += fmt(" c%u += kj_frames_in_word<%u>(r) << 16;", r, lay.kn);
        } else {
            tail = (r & 1u) ? fmt("c%u += __popc(r) << 16;", r >> 1) : fmt("c%u += __popc(r);", r >> 1);
        }
        em.stmts.push_back(Emitter::Stmt{em.deep(), "", e, tail});
    }
    em.emit_all();

    std::string s = kPrelude;
    s += fmt("\n// layout: n=%u g=%u cls=%u inner=%u outer=%u split=%u unit_frames_log2=%u programs=%u\n", n, lay.g, lay.cls,
             lay.inner, lay.outer, lay.split, lay.unit_frames_log2, G);
    s += fmt("extern \"C\" __global__ void __launch_bounds__(%u, %u) kripke_jit_scan(const KjParams p) {\n", threads, min_blocks);
    s += fmt("  __shared__ unsigned s_models[%u], s_frames[%u], s_best[%u];\n", G, G, G);
    s += "  const unsigned lane = threadIdx.x & 31u;\n";
    s += "  for (unsigned item = blockIdx.x; item < p.n_items; item += gridDim.x) {\n";
    s += "    const unsigned long long u0 = p.unit_begin + (unsigned long long)item * p.units_per_item;\n";
    s += "    const unsigned long long rem = p.unit_begin + p.unit_count - u0;\n";
    s += "    const unsigned item_units = rem < p.units_per_item ? (unsigned)rem : p.units_per_item;\n";
    s += "    __syncthreads();\n";
    s += fmt("    for (unsigned i = threadIdx.x; i < %uu; i += %uu) { s_models[i] = 0u; s_frames[i] = 0u; s_best[i] = 0xFFFFFFFFu; }\n", G, threads);
    s += "    __syncthreads();\n";
    s += fmt("    for (unsigned t0 = 0; t0 < item_units; t0 += %uu) {\n", threads);
    s += "      const unsigned warp_rel = t0 + (threadIdx.x & ~31u);\n";
    s += "      if (warp_rel >= item_units) continue;\n";
    s += "      const unsigned rel = warp_rel + lane;\n";
    s += "      const bool valid = rel < item_units;\n";
    s += "      const unsigned long long unit = u0 + (valid ? rel : 0u);\n";
    std::string decl_unit, decl_outer, decl_inner;
    // (the mask declarations depend on what the body used: emitted after the body is known)
    for (uint32_t b : em.bits.used_unit) decl_unit += fmt("      const unsigned mu%u = 0u - (unsigned)((unit >> %u) & 1ull);\n", b, b);
    if (lay.table) {
        decl_unit += fmt("      const unsigned long long frame = p.class_table[unit >> %u];\n", lay.split);
        for (uint32_t e : em.used_table) decl_unit += fmt("      const unsigned me%u = 0u - (unsigned)((frame >> %u) & 1ull);\n", e, e);
    }
    for (uint32_t b : em.bits.used_outer) decl_outer += fmt("      const unsigned mo%u = 0u - ((jo >> %u) & 1u);\n", b, b);
    if (!lay.nest_first) for (uint32_t b : em.bits.used_inner) decl_inner += fmt("      const unsigned mi%u = 0u - ((ji >> %u) & 1u);\n", b, b);
    s += decl_unit;
    s += "      // values that are fixed for the unit\n" + em.body[0];
    for (uint32_t r = 0; r < G; ++r) {
        if (packed && !has_f) { if (!(r & 1u)) s += fmt("      unsigned c%u = 0u;\n", r >> 1); continue; }
        s += fmt("      unsigned c%u = 0u;", r);
        if (has_f && !packed) s += fmt(" unsigned f%u = 0u;", r);
        s += "\n";
    }
    s += "#pragma unroll 1\n";
    s += fmt("      for (unsigned jo = 0; jo < %uu; ++jo) {\n", 1u << lay.outer);
    s += decl_outer;
    s += em.body[1];
    if (fmode == F_ANY) for (uint32_t r = 0; r < G; ++r) s += fmt("      unsigned a%u = 0u;\n", r);
    if (!lay.nest_first) {
        s += "#pragma unroll 1\n";
        s += fmt("      for (unsigned ji = 0; ji < %uu; ++ji) {\n", 1u << lay.inner);
        s += decl_inner;
        s += em.body[2];
        s += "      }\n";
    } else {
        // one loop over the nest_first slowest valuation bits, then a two-iteration loop per remaining bit, slower
        // bits outside: the body of a loop holds the values whose fastest-changing input is one of its bits
        const uint32_t rest = lay.inner - lay.nest_first;                    // single-bit loops
        s += "#pragma unroll 1\n";
        s += fmt("      for (unsigned js = 0; js < %uu; ++js) {\n", 1u << lay.nest_first);
        for (uint32_t b : em.bits.used_inner)
            if (b >= rest) s += fmt("      const unsigned mi%u = 0u - ((js >> %u) & 1u);\n", b, b - rest);
        s += em.body[2];
        for (uint32_t j = 0; j < rest; ++j) {
            const uint32_t b = rest - 1 - j;
            s += "#pragma unroll 1\n";
            s += fmt("      for (unsigned jb%u = 0; jb%u < 2u; ++jb%u) {\n", b, b, b);
            if (em.bits.used_inner.count(b)) s += fmt("      const unsigned mi%u = 0u - jb%u;\n", b, b);
            s += em.body[3 + j];
        }
        for (uint32_t j = 0; j <= rest; ++j) s += "      }\n";
    }
    if (fmode == F_ANY) for (uint32_t r = 0; r < G; ++r) s += packed ? fmt("      if (a%u != 0u) c%u += 65536u;\n", r, r) : fmt("      f%u += (a%u != 0u);\n", r, r);
    s += "      }\n";
    for (uint32_t r = 0; r < G; ++r) {
        const char *fm = fmode == F_MODELS ? "0" : fmode == F_THREAD ? "1" : "2";
        std::string c = fmt("c%u", r), f = has_f ? fmt("f%u", r) : std::string("0u");
        if (packed && has_f) { f = fmt("(c%u >> 16)", r); c = fmt("(c%u & 0xFFFFu)", r); }
        else if (packed) c = (r & 1u) ? fmt("(c%u >> 16)", r >> 1) : fmt("(c%u & 0xFFFFu)", r >> 1);
        s += fmt("      kj_flush<%u, %s>(%uu, ", lay.split, fm, r) + c + ", " + f + ", valid, warp_rel, lane, s_models, s_frames, s_best);\n";
    }
    s += "    }\n";
    s += "    __syncthreads();\n";
    s += fmt("    for (unsigned i = threadIdx.x; i < %uu; i += %uu)\n", G, threads);
    s += "      if (s_best[i] != 0xFFFFFFFFu) {\n";
    s += "        KjAccum *a = p.accum + p.slot_record[i];\n";
    s += "        atomicAdd(&a->models, (unsigned long long)s_models[i] << p.model_shift);\n";
    s += "        atomicAdd(&a->frames, (unsigned long long)s_frames[i]);\n";
    s += fmt("        atomicMin(&a->best, ((u0 + s_best[i]) >> %u) << %u);\n", lay.split, lay.unit_frames_log2);
    s += "      }\n";
    s += "  }\n}\n";
    {
        double per_word = 0;
        uint64_t emitted = 0;
        std::string by_level;
        for (int L = 0; L <= em.deep(); ++L) {
            per_word += (double)em.ops[L] * jit_level_weight(lay, L);
            emitted += em.ops[L];
            by_level += fmt(" %llu", (unsigned long long)em.ops[L]);
        }
        s += fmt("// graph nodes evaluated: box=%u and=%u; lop3 by loop level (unit, outer, inner bits slowest first):%s; per word %.1f\n",
                 em.n_box, em.n_and, by_level.c_str(), per_word);
        if (stats) {
            stats->logic_ops_emitted = emitted;
            stats->logic_ops_per_word = per_word;
            stats->n_box = em.n_box;
            stats->n_and = em.n_and;
        }
    }
    return s;
}

}  // namespace kripke
