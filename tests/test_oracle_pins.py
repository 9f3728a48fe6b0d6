"""Pins for the oracle (oracle/): values the paper prints, closed forms, invariants, brute force.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the
oracle (wrong index convention, transposed relation, swapped box/dia, wrong dead-end case, wrong
class filter, wrong witness order) fails at least one of them.  Citations: P:n = PAPER.md line n.
"""
import itertools
import json
import os

import numpy as np
import pytest

import workloads as W
from oracle import kripke_oracle as O

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))
K, T, S4, S5 = 0, 1, 2, 3


def prog(text):
    return W.to_postfix(W.parse(text))


AX = {name: W.to_postfix(t) for name, t in W.named_axioms().items()}


# ------------------------------------------------------------------------------------------
# A. the Python oracle against the paper and the mathematics
# ------------------------------------------------------------------------------------------
def test_py_prop5_certificate():
    """masks (2,4,8,16,32,0), world 0: alpha_2 holds, alpha_3 fails."""
    g = GOLD["prop5_certificate"]
    a2, a3 = W.to_postfix(W.alpha(2)), W.to_postfix(W.alpha(3))
    assert O.check_certificate(a3, g["n"], g["succ"], [], g["world"], K) is True
    assert O.check_certificate(a2, g["n"], g["succ"], [], g["world"], K) is False
    f = sum(s << (6 * w) for w, s in enumerate(g["succ"]))
    assert f == 541098242
    assert O.relation_from_index(6, f) == {(i, i + 1) for i in range(5)}
    assert O.check_pair_witness(a2, a3, 6, 0, K, f, 0, 0)
    # not reflexive, so it is no certificate for T
    assert O.check_certificate(a3, g["n"], g["succ"], [], g["world"], T) is False


@pytest.mark.parametrize("m", [1, 2, 3])
def test_py_lemma2_false_distances(m):
    """on the directed path of 2m+2 worlds, alpha_m is false exactly at r in {1,3,..,2m-1}."""
    n = 2 * m + 2
    R = {(i, i + 1) for i in range(n - 1)}
    for mm in (m, m + 1):
        ts = O.truth_set(n, R, [], W.alpha(mm))
        false_r = sorted(n - 1 - w for w in range(n) if w not in ts)
        assert false_r == list(range(1, 2 * mm, 2))
    # root: alpha_m true, alpha_{m+1} false
    assert O.sat(n, R, [], 0, W.alpha(m)) and not O.sat(n, R, [], 0, W.alpha(m + 1))


def test_py_dead_end_and_connectives():
    """P:215 'vacuously true at the dead end'; the connectives on a 2-world model by hand."""
    R = {(0, 1)}                       # 0 -> 1, 1 is a dead end
    V = [{1}, {0}]                     # p at world 1, q at world 0
    ts = lambda s: O.truth_set(2, R, V, W.parse(s))
    assert ts("[]F") == [1] and ts("<>T") == [0]
    assert ts("[]p") == [0, 1] and ts("<>p") == [0] and ts("[]q") == [1] and ts("<>q") == []
    assert ts("p&q") == [] and ts("p|q") == [0, 1] and ts("p->q") == [0] and ts("q->p") == [1]
    assert ts("~p") == [0] and ts("T") == [0, 1] and ts("F") == []


def test_py_index_conventions():
    """Readings R2, R3: edge w->u is bit w*n+u of f; p_i at w is bit i*n+w of v."""
    assert O.relation_from_index(3, 1 << (1 * 3 + 2)) == {(1, 2)}
    assert O.valuation_from_index(3, 2, 1 << (1 * 3 + 2)) == [set(), {2}]
    assert O.index_from_relation(3, {(2, 0), (0, 0)}) == (1 << 6) | 1


def _fo(n, R, name):
    """First-order conditions written out a second time, independently of oracle/ (test-side)."""
    W_ = range(n)
    if name == "reflexive":
        return all((w, w) in R for w in W_)
    if name == "serial":
        return all(any((w, u) in R for u in W_) for w in W_)
    if name == "transitive":
        return all((w, t) in R for w, u, t in itertools.product(W_, W_, W_) if (w, u) in R and (u, t) in R)
    if name == "euclidean":
        return all((u, t) in R for w, u, t in itertools.product(W_, W_, W_) if (w, u) in R and (w, t) in R)
    if name == "symmetric":
        return all((u, w) in R for (w, u) in R)
    if name == "partially_functional":
        return all(u == t for w, u, t in itertools.product(W_, W_, W_) if (w, u) in R and (w, t) in R)
    if name == "dense":
        return all(any((w, u) in R and (u, t) in R for u in W_) for (w, t) in R)
    if name == "confluent":
        return all(any((u, z) in R and (t, z) in R for z in W_)
                   for w, u, t in itertools.product(W_, W_, W_) if (w, u) in R and (w, t) in R)
    raise KeyError(name)


@pytest.mark.parametrize("axiom", ["T", "D", "4", "5", "B", "CD", "C4", "G"])
def test_py_table9_correspondence_n_le_3(axiom):
    """P:366-376 (Table 9): the axiom is frame-valid exactly on the frames with the condition."""
    cond = GOLD["table9"][axiom]
    phi = O.parse_postfix(AX[axiom])
    for n in (1, 2, 3):
        for f in range(1 << (n * n)):
            R = O.relation_from_index(n, f)
            valid = all(not O.refutes(n, R, O.valuation_from_index(n, 1, v), phi) for v in range(1 << n))
            assert valid == _fo(n, R, cond), (axiom, n, f)


def test_py_class_counts_and_order():
    cf = GOLD["closed_forms"]
    for n in (1, 2, 3):
        assert len(O.class_frames(n, K)) == 1 << (n * n)
        assert len(O.class_frames(n, T)) == cf["reflexive"][n - 1]
        assert len(O.class_frames(n, S4)) == cf["preorders"][n - 1]
        s5 = O.class_frames(n, S5)
        assert len(s5) == cf["equivalences"][n - 1]
        assert s5 == sorted(s5)
    # n=2 equivalences by hand: identity (bits 0,3) and the full relation
    assert O.class_frames(2, S5) == [0b1001, 0b1111]


def test_py_never_and_always_refuted():
    """K axiom and the tautology are refuted nowhere; F is refuted everywhere, and the
    first witness is (first frame of the class, valuation 0, world 0)."""
    for cls in (K, T, S4, S5):
        for n in (1, 2):
            assert O.census(AX["K"], n, 2, cls)[0] == 0
            assert O.census(prog("p->p"), n, 2, cls)[0] == 0
            frames = O.class_frames(n, cls)
            m, fr, wit = O.census(prog("p&~p"), n, 2, cls)
            assert (m, fr) == (len(frames) << (2 * n), len(frames))
            assert wit == (frames[0], 0, 0)
    assert O.census(AX["K"], 1, 2, K)[2] == (O.NO_WITNESS, 0, 0)


def test_py_witness_is_lexicographically_first():
    """[]p -> p at n=2: the first frame (f=0, no edges) refutes it with p false somewhere:
    v=0 (p nowhere) and world 0."""
    m, fr, wit = O.census(AX["T"], 2, 1, K)
    assert wit == (0, 0, 0)
    assert fr == 16 - 4                       # refuted on exactly the non-reflexive frames
    # in class T it is never refuted
    assert O.census(AX["T"], 2, 1, T)[0] == 0
    # <>T at n=2, class K: first refuting frame is f=0 (world 0 has no successor)
    assert O.census(prog("<>T"), 2, 0, K)[2] == (0, 0, 0)
    # []F -> F... p at n=2: refuted iff some world has p false; first (f,v) = (0,0), world 0
    assert O.census(prog("p"), 2, 1, K)[2] == (0, 0, 0)
    # q with k=2: v=0 refutes; and for 'p->q' the first refuting v has p true somewhere, q false there
    m, fr, wit = O.census(prog("p->q"), 2, 2, K)
    assert wit == (0, 1, 0)                   # v=1: p at world 0, q nowhere


# ------------------------------------------------------------------------------------------
# B. the C volume oracle against the Python oracle, closed forms and the paper
# ------------------------------------------------------------------------------------------
def test_c_equals_python_on_small_models(vol):
    """Brute force: counts and witnesses of C1 formulas, every class, n <= 3."""
    c1 = W.corpus_c1()
    sel = c1[:12] + [AX["K"], AX["4"], AX["5"], prog("[]<>p-><>[]q"), prog("<>(p&[]~q)|[]F")]
    code, offs = W.pack_programs(sel)
    for n in (1, 2, 3):
        for cls in (K, T, S4, S5):
            if n == 3 and cls == K:
                frames = None
                rng = (100, 40)              # a window is enough at n=3, K
            else:
                rng = (0, None)
            r = vol.census(code, offs, n, 2, cls, rng[0], rng[1])
            pyframes = O.class_frames(n, cls)
            for b, c in enumerate(sel):
                m, fr, wit = O.census(c, n, 2, cls, rng[0], rng[1], frames=pyframes)
                got = (int(r["models"][b]), int(r["frames"][b]),
                       (int(r["wit_f"][b]), int(r["wit_v"][b]), int(r["wit_w"][b])))
                assert got == (m, fr, wit), (n, cls, b)


def test_c_truth_equals_python_on_random_models(vol):
    rng = W.SplitMix64(99)
    forms = W.corpus_c4(40) + W.corpus_c2(40)
    for n in (4, 5, 6):
        for _ in range(60):
            c = forms[rng.below(len(forms))]
            f = rng.next_u64() & ((1 << (n * n)) - 1)
            v = rng.next_u64() & ((1 << (3 * n)) - 1)
            ts = O.truth_set(n, O.relation_from_index(n, f), O.valuation_from_index(n, 3, v),
                             O.parse_postfix(c))
            assert vol.truth(c, n, f, 3, v) == [1 if w in ts else 0 for w in range(n)]


def test_c_closed_form_counts(vol):
    cf = GOLD["closed_forms"]
    for n in range(1, 6):
        for name in ("reflexive", "symmetric", "serial", "partially_functional", "transitive"):
            assert vol.count_condition(n, name) == cf[name][n - 1], (n, name)
        assert len(vol.class_frames(n, T)) == cf["reflexive"][n - 1]
        assert len(vol.class_frames(n, S4)) == cf["preorders"][n - 1]
        assert len(vol.class_frames(n, S5)) == cf["equivalences"][n - 1]
    for n in (1, 2, 3):
        for cls in (T, S4, S5):
            assert vol.class_frames(n, cls).tolist() == O.class_frames(n, cls)
        for name in ("euclidean", "dense", "confluent", "transitive"):
            bm = vol.condition_bitmap(n, name)
            assert bm.tolist() == [int(_fo(n, O.relation_from_index(n, f), name)) for f in range(1 << (n * n))]
    assert sum(1 << (n * n) for n in range(1, 6)) == GOLD["frames_through_five"]["value"]


@pytest.mark.parametrize("axiom", ["T", "D", "4", "5", "B", "CD", "C4", "G"])
def test_c_table9_correspondence_n4(vol, axiom):
    """At n=4 the axiom is refuted on no frame with the condition and on every frame without it
    (frame-by-frame equality of the two extensions)."""
    cond = GOLD["table9"][axiom]
    bm = vol.condition_bitmap(4, cond)
    code, offs = W.pack_programs([AX[axiom]])
    yes = np.nonzero(bm)[0].astype(np.uint64)
    no = np.nonzero(bm == 0)[0].astype(np.uint64)
    assert int(vol.census_list(code, offs, 4, 1, yes)["frames"][0]) == 0
    assert int(vol.census_list(code, offs, 4, 1, no)["frames"][0]) == len(no)


def test_c_mckinsey_matches_no_library_condition(vol):
    """M = []<>p -> <>[]p has no match among the tested conditions (n <= 4)."""
    code, offs = W.pack_programs([AX["M"]])
    r = vol.census(code, offs, 4, 1)
    valid = (1 << 16) - int(r["frames"][0])
    assert all(valid != vol.count_condition(4, c) for c in vol.COND)


@pytest.mark.parametrize("axiom,cond", [("T", "reflexive"), ("B", "symmetric"), ("4", "transitive")])
def test_c_n5_validity_counts(vol, axiom, cond):
    """BASELINE.json north_star: []p->p valid on exactly the 2^(n^2-n) reflexive frames, []p->[][]p on
    the transitive ones, p->[]<>p on the 2^(n(n+1)/2) symmetric ones - here at n=5, full K range."""
    code, offs = W.pack_programs([AX[axiom]])
    r = vol.census(code, offs, 5, 1)
    assert (1 << 25) - int(r["frames"][0]) == GOLD["closed_forms"][cond][4]


def test_c_corpus_chain_44678_5621_frontier(vol):
    """P:143 / P:177 / P:145: 44,678 formulas -> 5,621 classes on models of <= 3 worlds; K frontier
    of the representatives 5,084 at one world, 536 at two, 1 never (p->p)."""
    g = GOLD["corpus_counts"]
    forms = W.enumerate_constant_free(7, 2)
    assert len(forms) == g["enumerated"]
    progs = [W.to_postfix(t) for t in forms]
    code, offs = W.pack_programs(progs)
    a, b = vol.signatures(code, offs, 3, 2)
    first = {}
    for i, s in enumerate(zip(a.tolist(), b.tolist())):
        first.setdefault(s, i)
    reps = [progs[i] for i in sorted(first.values())]
    assert len(reps) == g["classes_le3"]
    rc, ro = W.pack_programs(reps)
    at1 = vol.census(rc, ro, 1, 2)["models"] > 0
    at2 = vol.census(rc, ro, 2, 2)["models"] > 0
    at3 = vol.census(rc, ro, 3, 2)["models"] > 0
    assert int(at1.sum()) == g["frontier_1"]
    assert int((~at1 & at2).sum()) == g["frontier_2"]
    never = np.nonzero(~at1 & ~at2 & ~at3)[0]
    assert len(never) == g["unrefuted"]
    assert W.to_text(W.from_postfix(reps[never[0]])) == "(p->p)"
    assert int((~at1 & ~at2 & at3).sum()) == 0          # none needs three worlds


def test_c_alpha_pairs_separation_sizes(vol):
    """Table 3 and Prop. 5: (alpha_1, alpha_2) agree through 3 worlds, split at
    4; (alpha_2, alpha_3) agree through 5 and split at 6."""
    progs = [W.to_postfix(W.alpha(m)) for m in (1, 2, 3)]
    code, offs = W.pack_programs(progs)
    pairs = np.array([[0, 1], [1, 2]], dtype=np.uint32)
    for n in (1, 2, 3):
        r = vol.census(code, offs, n, 0, pairs=pairs)
        assert r["models"].tolist() == [0, 0] and r["wit_f"].tolist() == [vol.NO_WITNESS] * 2
    r4 = vol.census(code, offs, 4, 0, pairs=pairs)
    assert int(r4["models"][0]) > 0 and int(r4["models"][1]) == 0
    f, w = int(r4["wit_f"][0]), int(r4["wit_w"][0])
    assert O.check_pair_witness(progs[0], progs[1], 4, 0, K, f, 0, w)
    # regression values found with this oracle (SURVEY.md 8(c) scratch): 768 frames, first f=328
    assert (int(r4["frames"][0]), f, w) == (768, 328, 1)
    r5 = vol.census(code, offs, 5, 0, pairs=pairs)
    assert int(r5["models"][1]) == 0 and int(r5["frames"][0]) > 0
    # n=6: scan the prefix up to and including the first distinguishing frame
    first6 = 17335328                                   # SURVEY.md 8(c) scratch; re-derived here
    r6 = vol.census(code, offs, 6, 0, K, 0, first6 + 1, pairs=pairs[1:])
    assert (int(r6["frames"][0]), int(r6["wit_f"][0])) == (1, first6)
    assert O.check_pair_witness(progs[1], progs[2], 6, 0, K, first6, 0, int(r6["wit_w"][0]))
    # and the paper's own witness frame distinguishes them at world 0
    r = vol.census_list(code, offs, 6, 0, np.array([541098242], np.uint64), pairs=pairs[1:])
    assert (int(r["models"][0]), int(r["wit_w"][0])) == (1, 0)


def test_c_invariants(vol):
    """Duality, double negation, p<->q swap, class monotonicity, range additivity, weights."""
    c2 = W.corpus_c2(300)
    sub = [W.from_postfix(c) for c in c2[:40]]
    swap = lambda t: (t[0], 1 - t[1]) if t[0] == "var" else (t[0],) + tuple(swap(c) for c in t[1:])
    progs = []
    for t in sub:
        progs += [W.to_postfix(t), W.to_postfix(("not", ("not", t))), W.to_postfix(swap(t)),
                  W.to_postfix(("dia", t)), W.to_postfix(("not", ("box", ("not", t))))]
    code, offs = W.pack_programs(progs)
    r = vol.census(code, offs, 3, 2)
    m, fr = r["models"].reshape(-1, 5), r["frames"].reshape(-1, 5)
    assert (m[:, 0] == m[:, 1]).all() and (m[:, 0] == m[:, 2]).all() and (fr[:, 0] == fr[:, 2]).all()
    assert (m[:, 3] == m[:, 4]).all() and (r["wit_v"].reshape(-1, 5)[:, 3] == r["wit_v"].reshape(-1, 5)[:, 4]).all()
    code, offs = W.pack_programs(c2)
    per = [vol.census(code, offs, 3, 2, cls) for cls in (K, T, S4, S5)]
    for weaker, stronger in zip(per, per[1:]):
        assert (stronger["models"] <= weaker["models"]).all()
        assert ((stronger["models"] > 0) <= (weaker["models"] > 0)).all()
    a = vol.census(code, offs, 3, 2, K, 0, 200)
    b = vol.census(code, offs, 3, 2, K, 200, 312)
    assert (a["models"] + b["models"] == per[0]["models"]).all()
    assert (a["frames"] + b["frames"] == per[0]["frames"]).all()
    assert (np.minimum(a["wit_f"], b["wit_f"]) == per[0]["wit_f"]).all()
    fl = np.array([5, 17, 300], np.uint64)
    w1 = vol.census_list(code, offs, 3, 2, fl)
    w3 = vol.census_list(code, offs, 3, 2, fl, weights=np.array([3, 3, 3], np.uint64))
    assert (w3["models"] == 3 * w1["models"]).all() and (w3["frames"] == 3 * w1["frames"]).all()


def test_c_variable_complementation_invariance(vol):
    """v -> v XOR (worlds of p_i) is a bijection of the valuations of every frame, so phi(p, q), phi(~p, q) and
    phi(~p, ~q) have the same refuting-model count, refuting-frame count, first refuting frame and per-frame
    failure counts (what the CUDA path's canonical polarity relies on); the first valuation differs."""
    neg = lambda t, m: (("not", t) if (m >> t[1]) & 1 else t) if t[0] == "var" else (t[0],) + tuple(neg(c, m) for c in t[1:])
    sub = [W.from_postfix(c) for c in W.corpus_c2(400)[100:160]]
    progs = []
    for t in sub:
        progs += [W.to_postfix(t), W.to_postfix(neg(t, 1)), W.to_postfix(neg(t, 2)), W.to_postfix(neg(t, 3))]
    code, offs = W.pack_programs(progs)
    for n, cls in ((3, K), (4, T), (4, S4)):
        r = vol.census(code, offs, n, 2, cls)
        for key in ("models", "frames", "wit_f"):
            a = r[key].reshape(-1, 4)
            assert (a == a[:, :1]).all(), (n, cls, key)
        fc = vol.failure_counts(code, offs, n, 2, cls).reshape(len(sub), 4, -1)
        assert (fc == fc[:, :1, :]).all()
    v = vol.census(code, offs, 3, 2, K)["wit_v"].reshape(-1, 4)
    assert (v != v[:, :1]).any()


def test_c_filter_consistency(vol):
    """Counting over the class enumerator = counting over K restricted to class members."""
    c2 = W.corpus_c2(200)
    code, offs = W.pack_programs(c2)
    for cls, cond in ((T, ["reflexive"]), (S4, ["reflexive", "transitive"]),
                      (S5, ["reflexive", "transitive", "symmetric"])):
        bm = np.ones(1 << 9, dtype=bool)
        for c in cond:
            bm &= vol.condition_bitmap(3, c).astype(bool)
        viaK = vol.census_list(code, offs, 3, 2, np.nonzero(bm)[0].astype(np.uint64))
        viaC = vol.census(code, offs, 3, 2, cls)
        for key in viaK:
            assert (viaK[key] == viaC[key]).all()


@pytest.mark.parametrize("n", [2, 3, 4])
def test_c_validity_bitmaps_are_the_correspondents(vol, n):
    """Table 9 per frame: the validity bitmap of each Sahlqvist axiom over all K frames
    equals the bitmap of its first-order correspondent; K, p -> p and T are valid everywhere, F and
    p & ~p nowhere; validity = 'refuting_frames does not count this frame' of the census."""
    names = ["T", "4", "B", "D", "5", "CD", "C4", "G"]
    conds = ["reflexive", "transitive", "symmetric", "serial", "euclidean", "partially_functional", "dense",
             "confluent"]
    progs = [AX[a] for a in names] + [AX["K"], prog("p -> p"), prog("T"), prog("F"), prog("p & ~p")]
    code, offs = W.pack_programs(progs)
    val = vol.validity(code, offs, n, 2)
    assert val.shape == (len(progs), 1 << (n * n))
    for i, c in enumerate(conds):
        assert (val[i] == vol.condition_bitmap(n, c)).all(), names[i]
    assert val[8].all() and val[9].all() and val[10].all() and not val[11].any() and not val[12].any()
    res = vol.census(code, offs, n, 2)
    assert [int(x) for x in res["frames"]] == [int((1 << (n * n)) - v.sum()) for v in val]
    # class order: the T-class bitmap is the K bitmap restricted to the reflexive frames
    tf = vol.class_frames(n, T)
    assert (vol.validity(code, offs, n, 2, T) == val[:, tf.astype(np.int64)]).all()


def test_c_failure_counts_closed_forms_and_consistency(vol):
    """D_ij counts the (valuation, world) pairs where formula i fails on frame j.  Closed forms: F
    fails everywhere (n * 2^(kn)), T nowhere, p at half of the pairs; []F fails exactly at the worlds that
    have a successor, under every valuation; a count is 0 iff the frame is valid for the formula;
    the set-based oracle agrees pair by pair on two worlds; explicit relations = indexed frames."""
    n, k = 3, 2
    texts = ["F", "T", "p", "[]F", "[]p -> p", "p -> []<>p", "<>q & []p"]
    progs = [prog(t) for t in texts]
    code, offs = W.pack_programs(progs)
    cnt = vol.failure_counts(code, offs, n, k)
    pairs = n << (k * n)
    assert (cnt[0] == pairs).all() and (cnt[1] == 0).all() and (cnt[2] == pairs // 2).all()
    outdeg = np.array([sum(1 for w in range(n) if (f >> (w * n)) & 7) for f in range(1 << (n * n))])
    assert (cnt[3] == outdeg << (k * n)).all()
    assert ((cnt == 0) == vol.validity(code, offs, n, k).astype(bool)).all()
    for f in (0, 5, 17, 300, 511):
        R = O.relation_from_index(n, f)
        for b, c in enumerate(progs):
            phi = O.parse_postfix(c)
            want = sum(1 for v in range(1 << (k * n)) for w in range(n)
                       if not O.sat(n, R, O.valuation_from_index(n, k, v), w, phi))
            assert int(cnt[b, f]) == want
    rel = np.array([[[(f >> (w * n + u)) & 1 for u in range(n)] for w in range(n)] for f in range(1 << (n * n))], np.uint8)
    assert (vol.failure_counts(code, offs, n, k, rel=rel) == cnt).all()


# ------------------------------------------------------------------------------------------
# C. the isomorphism-orbit route (feeds tests/golden/n5_orbit.npz and c5_counts.npz:n5_frames)
# ------------------------------------------------------------------------------------------
def _relabel(n, pi, f):
    """Image of the K-index f under the world permutation pi (written a second time, in Python)."""
    g = 0
    for w in range(n):
        for u in range(n):
            if (f >> (w * n + u)) & 1:
                g |= 1 << (pi[w] * n + pi[u])
    return g


def _burnside_orbits(n):
    """Number of isomorphism classes of digraphs with loops on n labelled points by Burnside's lemma:
    (1/n!) sum over permutations of 2^(cycles of the induced permutation of the n*n ordered pairs)."""
    total = 0
    for pi in itertools.permutations(range(n)):
        seen, cycles = set(), 0
        for start in itertools.product(range(n), repeat=2):
            if start in seen:
                continue
            cycles += 1
            x = start
            while x not in seen:
                seen.add(x)
                x = (pi[x[0]], pi[x[1]])
        total += 2 ** cycles
    fact = 1
    for i in range(2, n + 1):
        fact *= i
    assert total % fact == 0
    return total // fact


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_c_orbits_counts_sizes_and_representatives(vol, n):
    """kov_orbits: the number of orbits is OEIS A000595 (2, 10, 104, 3,044, 291,968 - SURVEY 8(c)
    'relabelling invariance') and equals Burnside's count computed here; the sizes sum to 2^(n*n);
    every representative is the least member of its orbit and its size is the number of distinct
    relabellings (all orbits for n <= 3, a seeded sample for n = 4, 5); representatives ascend."""
    reps, sizes = vol.orbits(n)
    assert len(reps) == [2, 10, 104, 3044, 291968][n - 1] == _burnside_orbits(n)
    assert int(sizes.sum()) == 1 << (n * n)
    assert (np.diff(reps.astype(np.int64)) > 0).all()
    perms = list(itertools.permutations(range(n)))
    rng = W.SplitMix64(9100 + n)
    idx = range(len(reps)) if n <= 3 else sorted({rng.below(len(reps)) for _ in range(150)} | {0, len(reps) - 1})
    for i in idx:
        images = {_relabel(n, pi, int(reps[i])) for pi in perms}
        assert min(images) == int(reps[i]) and len(images) == int(sizes[i]), (n, i)
    # every frame belongs to exactly one listed orbit (n <= 3: all frames; n = 4, 5: seeded frames)
    repset = set(int(r) for r in reps)
    frames = range(1 << (n * n)) if n <= 3 else [rng.below(1 << (n * n)) for _ in range(300)]
    for f in frames:
        assert min(_relabel(n, pi, f) for pi in perms) in repset


def test_c_orbit_weighted_census_equals_direct_census(vol):
    """Relabelling invariance (P:123 scans labelled frames; the orbit route is the oracle's exact
    shortcut): class-K counts from one representative per orbit weighted by the orbit size equal the
    direct census over all labelled frames - all of C1 at n=3, 240 seeded C2 formulas at n=4 (only
    among non-constant ones), and the C5 pair counts at n=3, 4."""
    for progs, n in ((W.corpus_c1(), 3), (None, 4)):
        if progs is None:
            c2 = [c for c in W.corpus_c2() if (b"\x10" in c or b"\x11" in c)]
            rng = W.SplitMix64(9200)
            progs = [c2[i] for i in sorted({rng.below(len(c2)) for _ in range(260)})][:240]
        code, offs = W.pack_programs(progs)
        reps, sizes = vol.orbits(n)
        w = vol.census_list(code, offs, n, 2, reps, weights=sizes)
        d = vol.census(code, offs, n, 2, K)
        assert (w["models"] == d["models"]).all() and (w["frames"] == d["frames"]).all()
        assert d["models"].max() > 0 and (d["models"] != d["models"][0]).any()
    pprogs, pairs, _ = W.pairs_c5(300)
    code, offs = W.pack_programs(pprogs)
    pairs = np.array(pairs, np.uint32)
    for n in (3, 4):
        reps, sizes = vol.orbits(n)
        w = vol.census_list(code, offs, n, 0, reps, weights=sizes, pairs=pairs)
        d = vol.census(code, offs, n, 0, K, pairs=pairs)
        assert (w["frames"] == d["frames"]).all() and (w["models"] == d["models"]).all()


def test_py_distinguish_pinned_directly():
    """The Python pair path against things fixed outside it (it used to be compared only with
    distinguish_relations, which shares its formula):
    - by hand on one world: []p and <>p differ exactly on the dead-end frame (both valuations, at world 0) and
      coincide with p on the reflexive one;
    - p and ~p differ at every world of every model; a formula never differs from itself;
    - phi and T differ where phi fails, so the pair (phi, T) has the census of phi (pinned above by Table 9,
      closed forms and hand-computed cases), including the witness;
    - Table 3 / Prop. 5: alpha_1 and alpha_2 agree on every frame of <= 3 worlds and are
      split by a four-world frame; the first such frame is accepted by the certificate checker."""
    p, notp = prog("p"), prog("~p")
    assert O.distinguish(prog("[]p"), prog("<>p"), 1, 1) == (2, 1, (0, 0, 0))
    for n in (1, 2):
        frames = 1 << (n * n)
        assert O.distinguish(p, notp, n, 1) == (frames << n, frames, (0, 0, 0))
        assert O.distinguish(prog("[]p -> p"), prog("[]p -> p"), n, 1) == (0, 0, (O.NO_WITNESS, 0, 0))
    for text in ("[]p -> p", "p -> []<>p", "[](p -> q) -> ([]p -> []q)", "<>T"):
        k = 2 if "q" in text else (1 if "p" in text else 0)
        for cls in (K, T):
            assert O.distinguish(prog(text), prog("T"), 2, k, cls) == O.census(prog(text), 2, k, cls), (text, cls)
    a1, a2 = W.to_postfix(W.alpha(1)), W.to_postfix(W.alpha(2))
    for n in (1, 2, 3):
        assert O.distinguish(a1, a2, n, 0) == (0, 0, (O.NO_WITNESS, 0, 0))
    models, frames, (f, v, w) = O.distinguish(a1, a2, 4, 0)
    assert models == frames > 0 and v == 0                       # no variables: one valuation per frame
    assert (frames, f, w) == (768, 328, 1)                       # SURVEY.md 8(c) scratch; the C oracle finds the same
    assert O.check_pair_witness(a1, a2, 4, 0, K, f, v, w)
    assert all(not O.check_pair_witness(a1, a2, 4, 0, K, g, 0, u) for g in range(0, f, 37) for u in range(4))
