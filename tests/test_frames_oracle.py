"""Pins for the oracle's explicit-frame-list functions (oracle/kripke_oracle.py census_relations /
distinguish_relations, oracle/volume_oracle.c kov_census_relations) and for the seeded frame
generators.  No CUDA.  Citations: P:n = PAPER.md line n.
"""
import numpy as np
import pytest

import workloads as W
from oracle import kripke_oracle as O
from workloads import frames as F


def prog(text):
    return W.to_postfix(W.parse(text))


AX = {name: W.to_postfix(t) for name, t in W.named_axioms().items()}


@pytest.fixture(scope="module")
def vol():
    from oracle import volume
    volume.build()
    return volume


def dia_chain(m, base="T"):
    return prog("<>" * m + base)


def box_chain(m, base="F"):
    return prog("[]" * m + base)


# ------------------------------------------------------------------------------------------
# generators: shapes and the defining property of every template
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [6, 9, 16])
def test_templates_shape(n):
    names, rel = F.templates(n)
    assert rel.shape == (len(names), n, n) and rel.dtype == np.uint8
    t = dict(zip(names, rel))
    assert t["path"].sum() == n - 1 and all(t["path"][w, w + 1] for w in range(n - 1))
    assert (t["reverse_path"] == t["path"].T).all()
    assert t["reflexive_path"].sum() == 2 * n - 1 and t["reflexive_path"].trace() == n
    assert t["cycle"].sum() == n and t["cycle"][n - 1, 0] == 1
    assert t["star"][0].sum() == n - 1 and t["star"][1:].sum() == 0
    assert t["fork"][n - 3].sum() == 2 and t["fork"][n - 2:].sum() == 0
    assert t["complete"].sum() == n * n and t["empty"].sum() == 0
    # the six-world path is the certificate frame of Proposition 5 (masks 2,4,8,16,32,0)
    assert F.succ_masks(F.templates(6)[1])[0].tolist() == [2, 4, 8, 16, 32, 0]


def test_generators_are_seeded_and_in_range():
    for gen in (F.erdos_renyi, F.edge_flip, F.dead_end_insertion, F.back_edge_injection):
        a, b = gen(7, 300), gen(7, 300)
        assert a.shape == (300, 7, 7) and a.dtype == np.uint8 and a.max() <= 1
        assert (a == b).all()
    assert (F.dead_end_insertion(8, 200).sum(axis=2) == 0).any(axis=1).all()
    s = F.stress_list(10, 1000)
    assert s.shape == (1000, 10, 10)
    m = F.succ_masks(s)
    assert m.dtype == np.uint16 and m.shape == (1000, 10)
    j, w, u = 517, 3, 8
    assert ((int(m[j, w]) >> u) & 1) == s[j, w, u]


# ------------------------------------------------------------------------------------------
# the Python oracle on explicit frames
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("m", [1, 2, 3])
def test_py_lemma2_on_the_path_template(m):
    """P:213-215 (Lemma 2) and Table 3: on the directed path of 2m+2 worlds alpha_m and
    alpha_{m+1} differ exactly at the worlds at distance 2m+1 from the dead end, i.e. at the root."""
    n = 2 * m + 2
    a, b = W.to_postfix(W.alpha(m)), W.to_postfix(W.alpha(m + 1))
    models, frames, wit = O.distinguish_relations(a, b, n, 0, [F.path(n)])
    assert (models, frames, wit) == (1, 1, (0, 0, 0))
    # one world fewer: the two formulas agree everywhere on the shorter path
    assert O.distinguish_relations(a, b, n - 1, 0, [F.path(n - 1)])[0] == 0


def test_py_walk_length_closed_form():
    """<>^m T holds at w iff a walk of length m starts at w.  On the path of n worlds that is
    w <= n-1-m; on a cycle always; on the star only for m <= 1 at the centre.  (P:190 names
    <>^5 T / <>^6 T as an exact five-indistinguishable pair: they split on the six-world path.)"""
    for n in (6, 7, 9):
        for m in (1, 4, 5, 6):
            refuted_worlds = [w for w in range(n) if not (w <= n - 1 - m)]
            models, frames, wit = O.census_relations(dia_chain(m), n, 0, [F.path(n), F.cycle(n), F.star(n)])
            star_refuted = True                       # some leaf never has a successor
            assert models == (1 if refuted_worlds else 0) + 0 + (1 if star_refuted else 0)
            if refuted_worlds:
                assert wit == (0, 0, min(refuted_worlds))
    m, fr, wit = O.distinguish_relations(dia_chain(5), dia_chain(6), 6, 0, [F.cycle(6), F.star(6), F.path(6)])
    assert (m, fr, wit) == (1, 1, (2, 0, 0))
    # dual pair []^5 F / []^6 F: []^m F holds at w iff no walk of length m starts at w
    m, fr, wit = O.distinguish_relations(box_chain(5), box_chain(6), 6, 0, [F.reverse_path(6)])
    assert (m, fr, wit) == (1, 1, (0, 0, 5))


def test_py_list_census_equals_index_census():
    """The list route (matrices) and the index route (already pinned in test_oracle_pins.py) give the
    same counts and the same first witness when the list is 'all frames of n worlds in index order';
    catches a transposed matrix or a wrong position/witness convention."""
    n = 2
    mats = [[[(f >> (w * n + u)) & 1 for u in range(n)] for w in range(n)] for f in range(1 << (n * n))]
    for text in ["[]p -> p", "p -> []<>p", "[]p -> [][]p", "<>p -> []<>p", "[](p -> q) -> ([]p -> []q)", "<>T"]:
        k = 2 if "q" in text else (1 if "p" in text else 0)
        assert O.census_relations(prog(text), n, k, mats) == O.census(prog(text), n, k)
    assert O.distinguish_relations(prog("[]p"), prog("<>p"), n, 1, mats) == O.distinguish(prog("[]p"), prog("<>p"), n, 1)


# ------------------------------------------------------------------------------------------
# the C oracle on explicit frames
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,k,count", [(6, 1, 40), (7, 0, 120), (9, 1, 6), (12, 0, 60), (16, 0, 40)])
def test_c_equals_python_on_stress_lists(vol, n, k, count):
    rel = F.stress_list(n, count)
    atoms = "pT" if k else "TF"
    rng = W.SplitMix64(99 + n)
    forms = [W.gen_formula(rng, 9, 4, atoms) for _ in range(6)] + [W.alpha(2), W.alpha(3)]
    code, offs = W.pack_programs([W.to_postfix(t) for t in forms])
    res = vol.census_relations(code, offs, n, k, rel)
    for b, t in enumerate(forms):
        m, fr, wit = O.census_relations(W.to_postfix(t), n, k, rel)
        assert (int(res["models"][b]), int(res["frames"][b])) == (m, fr)
        assert (int(res["wit_f"][b]), int(res["wit_v"][b]), int(res["wit_w"][b])) == wit
    pairs = np.array([[0, 1], [6, 7], [2, 2]], np.uint32)
    pres = vol.census_relations(code, offs, n, k, rel, pairs=pairs)
    for j, (a, b) in enumerate(pairs):
        m, fr, wit = O.distinguish_relations(W.to_postfix(forms[a]), W.to_postfix(forms[b]), n, k, rel)
        assert (int(pres["models"][j]), int(pres["frames"][j])) == (m, fr)
        assert (int(pres["wit_f"][j]), int(pres["wit_v"][j]), int(pres["wit_w"][j])) == wit


@pytest.mark.parametrize("n", [6, 8])
def test_c_correspondence_on_random_relations(vol, n):
    """Table 9 as a pin at sizes the exhaustive scan cannot reach: on any frame list,
    []p -> p is refuted exactly on the non-reflexive frames, []p -> [][]p on the non-transitive,
    p -> []<>p on the non-symmetric, []p -> <>p on the non-serial ones.  The first-order side is
    computed here with numpy, not by the oracle."""
    rel = np.concatenate([F.stress_list(n, 600), F.erdos_renyi(n, 300, densities=(0.9, 0.97)),
                          F.reflexive_path(n)[None], F.complete(n)[None]])
    # symmetric / transitive closures of some of them so the properties really occur
    sym = rel[:200] | rel[:200].transpose(0, 2, 1)
    tr = rel[200:400].copy()
    for _ in range(4):
        tr = ((tr.astype(np.int32) @ tr.astype(np.int32) > 0) | (tr > 0)).astype(np.uint8)
    rel = np.concatenate([rel, sym, tr])
    r32 = rel.astype(np.int32)
    refl = np.array([m.diagonal().all() for m in rel])
    trans = np.array([((a @ a > 0) <= (a > 0)).all() for a in r32])
    symm = np.array([(a == a.T).all() for a in rel])
    serial = (rel.sum(axis=2) > 0).all(axis=1)
    assert 0 < trans.sum() < len(rel) and 0 < symm.sum() < len(rel) and 0 < refl.sum() < len(rel)
    code, offs = W.pack_programs([AX["T"], AX["4"], AX["B"], AX["D"], AX["K"]])
    res = vol.census_relations(code, offs, n, 2, rel)
    want = [(~refl), (~trans), (~symm), (~serial), np.zeros(len(rel), bool)]
    for b, cond in enumerate(want):
        assert int(res["frames"][b]) == int(cond.sum())
        first = int(np.argmax(cond)) if cond.any() else O.NO_WITNESS
        assert int(res["wit_f"][b]) == first
    assert int(res["models"][4]) == 0            # K axiom: refuted on no model


def test_c_alpha_3_4_separate_at_eight_worlds(vol):
    """Table 3: (alpha_3, alpha_4) separate at 8 worlds - on the path template - and on no
    shorter path; the separating world is the root (Lemma 2)."""
    code, offs = W.pack_programs([W.to_postfix(W.alpha(m)) for m in (1, 2, 3, 4)])
    pairs = np.array([[0, 1], [1, 2], [2, 3]], np.uint32)
    for n in range(1, 11):
        res = vol.census_relations(code, offs, n, 0, F.path(n)[None], pairs=pairs)
        assert [int(x) for x in res["models"]] == [int(n >= 4), int(n >= 6), int(n >= 8)]
