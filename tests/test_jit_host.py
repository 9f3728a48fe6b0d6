"""Host side of the compiled scans (csrc/jit_dag.cpp, jit_emit.cpp, jit_runtime.cpp), no GPU needed:
the batch graph's rewrites are exact (truth sets equal the oracle's on random models), and the emitted
CUDA C compiles for sm_100a with NVRTC for every layout kind."""
import re

import numpy as np
import pytest

import workloads as W
from paper_2606_15437_b200 import binding as kb

K, T, S4, S5 = 0, 1, 2, 3


def _models(rng, n, k, count):
    out = []
    for _ in range(count):
        f = rng.next_u64() & ((1 << (n * n)) - 1)
        v = rng.next_u64() & ((1 << (k * n)) - 1)
        succ = [(f >> (w * n)) & ((1 << n) - 1) for w in range(n)]
        vals = [(v >> (i * n)) & ((1 << n) - 1) for i in range(k)]
        out.append((f, v, succ, vals))
    return out


def test_batch_graph_truth_equals_oracle(vol):
    """kripke_debug_dag_truth: the truth set a program's graph computes - after negation edges, the and / box
    normal form, flattened and sorted conjunctions, box x & box y = box (x & y), constant folding and the
    canonical variable order - equals the oracle's truth set on random models (n = 3, 5, 6; k = 0..3)."""
    rng = W.SplitMix64(77001)
    sets = [(W.corpus_c1(250), 2), (W.corpus_c2(900)[500:], 2), (W.corpus_c4(250), 3), (W.pairs_c5(120)[0], 0)]
    sets.append(([W.to_postfix(t) for t in W.named_axioms().values()], 2))
    extra = ["[]p & []q", "[]p & ([]q & []~p)", "<>p | <>q", "~([]p & []q) | [](q & p)", "(p & q) & (q & p)",
             "p & ~p", "[](p | ~p)", "<>(p & ~p)", "[]([]p & []q) -> [][](p & q)", "(q -> p) & (q | p)"]
    sets.append(([W.to_postfix(W.parse(t)) for t in extra], 2))
    for progs, k in sets:
        for c in progs:
            for n in (3, 5, 6):
                for f, v, succ, vals in _models(rng, n, k, 3):
                    want = sum(b << w for w, b in enumerate(vol.truth(c, n, f, k, v)))
                    got = kb.debug_dag_truth(c, k, n, succ, vals)
                    assert got == want, (W.to_text(W.from_postfix(c)), n, f, v)


@pytest.mark.parametrize("flags", [0, kb.NO_GUARDED_ROOTS, kb.NO_BOX_DISTRIBUTION])
def test_evaluation_forms_refute_exactly_the_oracles_models(vol, flags):
    """kripke_debug_batch_refuted: the forms the compiled kernels evaluate - the refutation test pushed through the
    conjunctions and boxes at the top of each formula (guard sets S_d = worlds reachable in exactly d steps) and box
    redistributed over conjunctions by the batch's cost - refute exactly the models the oracle's truth set
    refutes, for every formula of a batch on random models (classes K and T, n = 3..6), and rewrites do happen."""
    rng = W.SplitMix64(77002)
    extra = ["[]p", "[][]p", "[](p & q)", "[]p & []q", "[][](p -> q) & p", "[]F", "[][]F", "[]T", "[]([]p & q)",
             "[]([]F | p)", "[]p & ([]q & ~[](p & q))", "[](p & []q) -> [](q & []p)", "<>p -> []<>p", "[](p & q & []p)"]
    sets = [(W.corpus_c2(700), 2), (W.corpus_c1(300) + [W.to_postfix(W.parse(t)) for t in extra], 2),
            (W.corpus_c4(200), 3), (W.pairs_c5(150)[0], 0)]
    total_rewrites = 0
    for progs, k in sets:
        code, offs = W.pack_programs(progs)
        for n, cls in ((3, K), (5, K), (5, T), (4, T), (6, K)):
            if n * n + k * n > 61:
                continue
            for f, v, succ, vals in _models(rng, n, k, 4):
                if cls == T:
                    f |= sum(1 << (w * n + w) for w in range(n))
                    succ = [(f >> (w * n)) & ((1 << n) - 1) for w in range(n)]
                got, rewrites = kb.debug_batch_refuted(code, offs, k, n, cls, succ, vals, flags)
                total_rewrites += rewrites
                for i, c in enumerate(progs):
                    want = not all(vol.truth(c, n, f, k, v))
                    assert bool(got[i]) == want, (W.to_text(W.from_postfix(c)), n, cls, f, v)
    assert (total_rewrites > 0) == (not (flags & kb.NO_BOX_DISTRIBUTION))


def test_guarded_roots_drop_the_top_boxes():
    """A formula that is a box of a variable costs n instructions per word in guarded form (no box is evaluated),
    n^2 + the test when its full truth set is computed."""
    code, offs = W.pack_programs([W.to_postfix(W.parse("[][](p | q)"))])
    guarded = kb.debug_jit_source(code, offs, 2, 5, K, 2)[2]
    plain = kb.debug_jit_source(code, offs, 2, 5, K, 2, 0, kb.NO_GUARDED_ROOTS)[2]
    assert guarded <= 12 and plain >= 3 * guarded and plain >= 30


def test_box_distribution_shares_nodes():
    """[]p & []q and [](p & q) are the same graph node; alpha-equivalent programs coincide after the
    canonical renaming (one compiled program for the two of them)."""
    a = [W.to_postfix(W.parse(t)) for t in ("[]p & []q", "[](q & p)", "[]q & []p")]
    code, offs = W.pack_programs(a)
    src, nk, ops, _ = kb.debug_jit_source(code, offs, 2, 5, K, 2)
    assert nk == 1 and "programs=1" in src
    b = [W.to_postfix(W.parse(t)) for t in ("[]p -> q", "[]q -> p", "<>p & []q", "[]p & <>q")]
    code, offs = W.pack_programs(b)
    src, nk, ops, _ = kb.debug_jit_source(code, offs, 2, 5, K, 2)
    assert "programs=2" in src


@pytest.mark.parametrize("n,k,cls", [(5, 2, K), (5, 2, T), (5, 2, S4), (5, 1, K), (5, 1, T), (5, 1, S5), (5, 0, K),
                                     (5, 0, T), (4, 2, K), (4, 1, K), (4, 0, K), (3, 2, K), (3, 1, T), (6, 0, K),
                                     (6, 1, K), (6, 2, K), (5, 3, K), (5, 3, T), (4, 3, S4), (2, 2, K)])
def test_emitted_kernels_compile_for_sm100a(n, k, cls):
    """Every layout kind (frames in the lanes, in the word loop, one thread per frame, several threads per
    frame, class-T diagonal, S4 / S5 table) compiles with NVRTC --gpu-architecture=sm_100a."""
    progs = {0: W.pairs_c5(60)[0], 1: [c for c in W.corpus_c4(400) if b"\x11" not in c and b"\x12" not in c][:40],
             2: W.corpus_c2(120), 3: W.corpus_c4(80)}[k]
    code, offs = W.pack_programs(progs)
    seen = 0
    for g in range(k + 1):
        r = kb.debug_jit_source(code, offs, k, n, cls, g, 0, compile=True)
        if r is None:
            continue
        src, nk, ops, cubin = r
        if nk == 0:
            continue
        seen += 1
        assert cubin > 0 and (ops > 0 or g < k)
        m = re.search(r"layout: n=(\d+) g=(\d+) cls=(\d+) inner=(\d+) outer=(\d+) split=(\d+) unit_frames_log2=(\d+)", src)
        assert m and int(m.group(1)) == n and int(m.group(2)) == g
        inner, outer, split, ufl = (int(m.group(i)) for i in (4, 5, 6, 7))
        kn = g * n
        # the loop and the unit cover the valuation bits exactly; a unit never mixes frames and frame parts
        assert (kn >= 5 and inner + split == kn - 5) or (kn < 5 and inner == split == 0)
        assert split == 0 or (outer == 0 and ufl == 0)
    assert seen >= 1
    # pairs compile as well
    pairs = np.array([[i, i + 1] for i in range(0, min(len(progs), 40) - 1, 2)], np.uint32)
    r = kb.debug_jit_source(code, offs, k, n, cls, k, 0, pairs=pairs, compile=True)
    assert r is None or r[1] == 0 or r[3] > 0


def test_no_layout_for_tiny_shapes():
    code, offs = W.pack_programs(W.pairs_c5(10)[0])
    assert kb.debug_jit_source(code, offs, 0, 2, K, 0) is None          # 16 models: less than one word
    assert kb.debug_jit_source(code, offs, 0, 5, S4, 0) is None         # table class needs the lanes for valuations


@pytest.mark.parametrize("n,k,cls", [(5, 2, K), (5, 2, T), (5, 2, S4), (3, 2, K), (5, 0, K), (6, 0, K), (4, 0, T),
                                     (5, 1, K), (4, 3, K)])
def test_density_kernels_compile_for_sm100a(n, k, cls):
    """The failure-density kernels (one frame per thread; one frame per lane with bit-plane counts) compile."""
    progs = {0: W.pairs_c5(40)[0], 1: [c for c in W.corpus_c4(400) if b"\x11" not in c and b"\x12" not in c][:30],
             2: W.corpus_c2(80), 3: W.corpus_c4(40)}[k]
    code, offs = W.pack_programs(progs)
    seen = 0
    for g in range(k + 1):
        r = kb.debug_jit_source(code, offs, k, n, cls, g, 0, compile=True, density=True)
        if r is None or r[1] == 0:
            continue
        seen += 1
        assert r[3] > 0 and "density layout" in r[0]
        body = r[0].split("density layout")[1]
        # no variables: one frame per lane, counts leave as bit planes (staged through shared memory when
        # the warp's words are consecutive, else unpacked per lane)
        assert ("KJ_CNT3" in body or "s_stage" in body) == (g == 0)
    assert seen >= 1
