// jit.h - compiled bit-sliced scans: the batch's programs become straight-line sm_100a code.
//
// The interpreted bit-sliced kernel (scan_sliced.cuh) spends a third of its issue slots on micro-op
// dispatch and evaluates every program on its own.  A batch is known when it is staged, so this path
// (1) turns the whole batch into ONE directed acyclic graph of distinct subterms (jit_dag.cpp:
//     negation is an edge attribute, or / imp / dia are rewritten onto and / box, conjunctions are
//     flattened and sorted, variables are renamed to a canonical order) - a subterm that occurs in
//     many formulas is evaluated once per 32-model word;
// (2) emits CUDA C for groups of programs (jit_emit.cpp): one kernel per group, a thread owns one
//     scan unit, loops over its 32-model words, and every node of the group's graph is a handful of
//     3-input logic instructions on named registers - no dispatch, no stack, no program memory;
// (3) compiles the groups with NVRTC for sm_100a and loads them (jit_runtime.cpp), cached per
//     process by source hash.
// The semantics are those of scan_sliced.cuh (Lemma 1 applied to 32 models at once);
// the reduction is the same warp -> block -> one global atomic triple per (block, program)
// (PAPER.md:74); witnesses are completed by finish_kernel.
#pragma once
#include <stdint.h>

#include <array>
#include <map>
#include <string>
#include <vector>

#include "internal.h"

namespace kripke {

// ---- the batch graph (jit_dag.cpp) ----------------------------------------------------------------
// A literal is node * 2 + neg.  Node kinds: the constant "false", a variable, and(a, b), box(a).
struct DagNode {
    enum Kind : uint8_t { CONST0, VAR, AND, BOX } kind;
    uint8_t var;            // VAR: index in the group's valuation
    uint32_t a, b;          // operand literals (AND: a < b)
    uint32_t salt;          // 0, or the owner record + 1 when subterm sharing is off
    uint8_t rank;           // loop level of the variables below it (not part of the node's identity)
};

struct Dag {
    std::vector<DagNode> nodes;
    uint32_t lit_const(bool v);
    uint32_t lit_var(uint32_t i);
    uint32_t mk_and(uint32_t x, uint32_t y);
    uint32_t mk_box(uint32_t x);
    // Postfix program -> literal.  rename: variable index -> index in the group's valuation; neg_mask: bit v =
    // variable v (as written) is read complemented.
    uint32_t build(const uint8_t *code, uint32_t len, const uint8_t *rename, uint32_t neg_mask = 0);
    // Variables a literal's cone mentions (bit i).
    uint32_t support(uint32_t lit) const;
    // Truth set (n-bit mask) of a literal on one model: succ[w] successor masks, val[i] variable masks.
    uint32_t eval(uint32_t lit, uint32_t n, const uint32_t *succ, const uint32_t *val) const;
    uint32_t salt = 0;      // applied to new AND / BOX nodes
    // Canonical graphs (the default) rewrite box x & box y into box (x & y) and order conjuncts by literal.  An
    // implementation graph (jit_opt.cpp) keeps conjunctions of boxes as they are and folds the conjuncts of low
    // loop level first (var_rank[i] = level of variable i), so that loop-invariant partial conjunctions are hoisted.
    bool merge_boxes = true;
    std::vector<uint8_t> var_rank;
    uint8_t rank_of(uint32_t lit) const { return nodes[lit >> 1].rank; }
    // Canonical text of a literal's cone (conjunctions flattened, operands sorted by text).
    std::string text(uint32_t lit) const;
  private:
    uint32_t intern(const DagNode &nd);
    void conjuncts(uint32_t lit, std::vector<uint32_t> *out) const;
    std::map<std::array<uint32_t, 5>, uint32_t> index_;
};

// Canonical variable order of one program (or pair): among the permutations of the variables it mentions, the one
// whose graph does the least work inside the loops (loop_var_mask: bit i = renamed variable i changes inside a
// thread's word loop on the layout in use; a subterm over the other variables is evaluated once per unit), ties
// broken by the least canonical text.  The choice depends on the alpha-equivalence class only, so alpha-equivalent
// programs get the same graph.  support_mask: variables mentioned; rename_out[v] = index in the reduced valuation.
// neg_out (may be null): also the variables to complement - v -> v XOR (the worlds of p_i) is a bijection of the
// valuations of every frame, so phi(p) and phi(~p) have the same refuting-model and refuting-frame counts, the
// same first refuting frame and the same failure densities; with neg_out the canonical form is taken over
// permutations and complementations, and more programs of a batch coincide.
void canonical_rename(const uint8_t *code_a, uint32_t len_a, const uint8_t *code_b, uint32_t len_b,
                      uint32_t support_mask, uint32_t n, uint32_t loop_var_mask, uint8_t *rename_out,
                      uint32_t *neg_out = nullptr);

// ---- cost-driven redistribution of box over conjunction (jit_opt.cpp) -------------------------------
struct JitLayout;
struct JitRoot;
struct JitOptStats {
    uint32_t rewrites = 0;
    double cost_before = 0, cost_after = 0;   // logic instructions per 32-model word of the needed graph nodes
};
// box (x1 & ... & xk) = box (S1) & ... & box (Sm) for every partition of the conjuncts, on every frame.  Which
// side is cheaper depends on what else the batch evaluates: the left side costs one box (n^2 instructions per
// word), the right side m boxes - but only those that no other formula needs anyway, and only at the loop level
// of their own variables.  Starting from the canonical graph (left sides only), applies the rewrite with the
// largest saving until none is left.  *roots is replaced by the roots in *out.
void jit_optimize(const Dag &in, const JitLayout &lay, std::vector<JitRoot> *roots, Dag *out, JitOptStats *stats);

// ---- layout (jit_emit.cpp) ------------------------------------------------------------------------
// Model index X = (class-order frame index << g*n) | v.  Bits 0..4 of X vary inside a word, the next
// `inner` bits (valuation) and `outer` bits (frame) are the thread's word loop, the rest is the
// thread's unit index; `split` = log2 threads per frame when a frame's valuations exceed the loop.
struct JitLayout {
    uint32_t n = 0, g = 0, cls = 0;
    uint32_t kn = 0;               // g * n
    uint32_t inner = 0, outer = 0, split = 0;
    uint32_t unit_frames_log2 = 0; // frames per unit = 2^this (0 when a unit is one frame or part of it)
    uint32_t lane_bits = 0;        // density kernels, one frame per lane: bits 5.. of X taken from the thread's lane
                                   // (= the low bits of its unit index), so that a warp's words are consecutive
    bool table = false;            // frames come from the class table (S4 / S5)
    uint32_t nest_first = 0;       // 0: the inner loop is one loop.  Else it is a nest: one loop over the nest_first slowest
                                   // valuation bits, then a two-iteration loop for each remaining bit, slower bits outside:
                                   // a value that depends only on slow bits is computed in the loop of the fastest bit it
                                   // depends on (levels 2 .. 2 + inner - nest_first), not once per word
};
// Is there a compiled layout for (n, g, class)?  Fills *out.
bool jit_layout(uint32_t n, uint32_t g, uint32_t cls, JitLayout *out);

// Loop level at which a bit of the model index changes in a thread (0 = fixed for the unit, 1 = outer loop,
// 2 = inner loop; nested layouts: 2 for the nest_first slowest bits of the inner loop, then one level per bit) for "p_i at world w" and for the edge w -> u (0 where the edge is no index bit: class T's
// diagonal, the table classes), and the cost of one instruction at a level per 32-model word.
int jit_atom_level(const JitLayout &lay, uint32_t var, uint32_t w);
int jit_edge_level(const JitLayout &lay, uint32_t w, uint32_t u);
double jit_level_weight(const JitLayout &lay, int level);

// One record of a group: a single formula (b == UINT32_MAX) or a pair.
//
// A single formula may be given in guarded form instead of by its root literal: a model refutes it iff its truth
// set is not W, i.e. iff the root fails at some world.  A positive conjunction fails somewhere iff one
// conjunct does, and box x fails somewhere iff x fails at a world that has a predecessor, so the
// test is pushed through the positive conjunctions and boxes at the top of the formula:
//     refuted  <=>  OR over (depth, lit) in guarded of  OR_u ( S_depth[u] & ~lit[u] ),
// S_0 = W, S_(d+1) = the successors of S_d - sets that depend on the frame only and are shared by every record.
// The boxes at the top of a formula are then never evaluated (n instructions per obligation instead of n^2 per box).
struct JitGuarded {
    uint32_t depth, lit;
    bool operator<(const JitGuarded &o) const { return depth != o.depth ? depth < o.depth : lit < o.lit; }
    bool operator==(const JitGuarded &o) const { return depth == o.depth && lit == o.lit; }
};
struct JitRoot {
    uint32_t a = 0, b = UINT32_MAX;        // literals (a is unused when guarded is not empty)
    std::vector<JitGuarded> guarded;
    // every literal whose value the record reads
    template <class F> void for_each_lit(F f) const {
        if (!guarded.empty()) { for (const JitGuarded &g : guarded) f(g.lit); return; }
        f(a);
        if (b != UINT32_MAX) f(b);
    }
    template <class F> void map_lits(F f) {
        if (!guarded.empty()) { for (JitGuarded &g : guarded) g.lit = f(g.lit); return; }
        a = f(a);
        if (b != UINT32_MAX) b = f(b);
    }
};
// Rewrites the single-formula roots into guarded form (pairs and roots that are a bare literal stay as they are).
void jit_guard_roots(const Dag &dag, std::vector<JitRoot> *roots);
// Does the model (succ[w] successor masks, val[i] variable masks) refute the record, evaluated as the compiled
// kernels evaluate it?  (host check of the guarded form and of the optimised graph)
bool jit_root_refuted(const Dag &dag, const JitRoot &root, uint32_t n, const uint32_t *succ, const uint32_t *val);

struct JitEmitStats {
    double logic_ops_per_word = 0;     // 3-input logic instructions executed per 32-model word: statements of the
                                       // inner loop + those of the outer loop and of the unit set-up per word
    uint64_t logic_ops_emitted = 0;    // statements' logic instructions, wherever they are placed
    uint32_t n_box = 0, n_and = 0;     // graph nodes evaluated per word (summed over kernels)
};

// Layout of the failure-density kernels: a thread owns whole frames (one frame and all its valuation words, or -
// no variables - 32 frames per word), so that it can write the per-frame counts itself.
bool jit_density_layout(uint32_t n, uint32_t g, uint32_t cls, JitLayout *out);

enum : uint32_t {
    JIT_MODE_SCAN = 0,      // per program: refuting models / frames, least refuting unit (Algorithm 1's outputs)
    JIT_MODE_DENSITY = 1    // per (program, frame): the number of (valuation, world) pairs that fail
};

// CUDA C source of one kernel `kripke_jit_scan` that evaluates roots[0..) on the layout.
std::string jit_emit_kernel(const Dag &dag, const JitLayout &lay, const std::vector<JitRoot> &roots,
                            uint32_t threads, uint32_t min_blocks, uint32_t mode, JitEmitStats *stats);

// Partition of the roots into kernels of at most `max_roots` that share as many subterms as possible.
std::vector<std::vector<uint32_t>> jit_partition(const Dag &dag, const std::vector<JitRoot> &roots,
                                                 const JitLayout &lay, uint32_t max_roots);
// Logic instructions per 32-model word the emitter generates for every node of the graph on this layout (a node
// that does not change inside the loops is charged its share of a word).
std::vector<double> jit_node_costs(const Dag &dag, const JitLayout &lay);

// ---- runtime (jit_runtime.cpp) --------------------------------------------------------------------
struct JitKernel {
    void *kernel = nullptr;        // cudaKernel_t
    uint32_t slot_base = 0;        // first slot (index into the group's slot_record)
    uint32_t n_slots = 0;
};

struct JitGroupPlan {
    JitLayout lay;
    std::vector<JitKernel> kernels;
    uint32_t *d_slot_record = nullptr;   // device: record per slot
    std::vector<uint32_t> h_slot_record; // the same on the host (a cached plan is re-uploaded from it)
    // density plans: program (slot) s writes the rows h_rows[h_row_begin[s] .. h_row_begin[s+1]) - its own record and
    // the records whose program it is (equal graphs under the canonical variable order and polarity)
    std::vector<uint32_t> h_row_begin, h_rows;
    uint32_t *d_row_begin = nullptr, *d_rows = nullptr;
    uint32_t n_slots = 0;
    uint32_t threads = 128;
    JitEmitStats stats;
    void release();
};

// Compiles (or fetches from the process cache) the kernels of one group.  Sources are compiled in
// parallel host threads.  Returns 0, a negative kripke_status, or a positive cudaError_t;
// *log_out receives the NVRTC log on a compile error.
int jit_build_group(const Dag &dag, const JitLayout &lay, const std::vector<JitRoot> &roots,
                    const std::vector<uint32_t> &slot_record, uint32_t max_roots, uint32_t min_blocks,
                    uint32_t mode, JitGroupPlan *out, std::string *log_out);

// Device copy of plan->h_slot_record (a plan taken from the process-wide cache owns no device memory yet).
int jit_upload_slots(JitGroupPlan *plan);

// Output of the density kernels: counts[record * total_frames + (class-order frame index - frame_base)].
struct JitDensityOut {
    uint32_t *counts;
    uint64_t total_frames, frame_base;
};

// Enqueues the group's kernels over the aligned class range of `job` (job.k = the group's g).
int jit_launch_group(const ScanJob &job, const JitGroupPlan &plan, uint32_t model_shift, const JitDensityOut *density,
                     void *stream, uint32_t *launches);

// Compiles one source to a cubin without loading it (tests on a box without a GPU): 0 or error.
int jit_compile_only(const std::string &source, std::string *log_out, size_t *cubin_bytes);
// Unloads every compiled module of the process-wide cache and forgets it; returns how many there were.  Only
// safe when no plan that holds one of their kernels can be launched again and none is running (api.cpp checks).
size_t jit_cache_clear();
size_t jit_cache_modules();

}  // namespace kripke
