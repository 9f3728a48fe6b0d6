"""Parity of the frame-list mode (kripke_eval_frames / kripke_distinguish_pairs_frames, through the C
ABI) with the oracle on the same seeded frame lists: bit-exact counts and witnesses, every witness
re-verified by the set-based checker.  P:n = PAPER.md line n.
"""
import numpy as np
import pytest

import workloads as W
from oracle import kripke_oracle as O
from workloads import frames as F

pytestmark = pytest.mark.gpu

KEYS = ("models", "frames", "wit_f", "wit_v", "wit_w")


@pytest.fixture(scope="module")
def kb():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2606_15437_b200 import binding
    binding.load()
    return binding


def dev_succ(rel):
    import torch
    m = F.succ_masks(rel)
    return torch.from_numpy(m.view(np.int16).reshape(-1).copy()).cuda()


def same(got, want, what=""):
    for key in KEYS:
        g, w = np.asarray(got[key]).astype(np.uint64), np.asarray(want[key]).astype(np.uint64)
        bad = np.nonzero(g != w)[0]
        assert len(bad) == 0, f"{what}: {key} differs at {bad[:5]}: got {g[bad[:5]]} want {w[bad[:5]]}"


def formulas(seed, count, k, budget=9, depth=4):
    rng = W.SplitMix64(seed)
    atoms = {0: "TF", 1: "pTF", 2: "pqTF"}[k]
    return [W.to_postfix(W.gen_formula(rng, budget, depth, atoms)) for _ in range(count)]


def certify(progs, res, n, k, rel, pairs=None):
    """Definition 1: the reported (frame, valuation, world) falsifies the formula (or is a
    disagreement world of the pair) for the set-based checker."""
    for b in range(len(res["models"])):
        j = int(res["wit_f"][b])
        if j == O.NO_WITNESS:
            assert int(res["models"][b]) == 0
            continue
        R = O.relation_from_matrix(n, rel[j])
        V = O.valuation_from_index(n, k, int(res["wit_v"][b]))
        w = int(res["wit_w"][b])
        if pairs is None:
            assert not O.sat(n, R, V, w, O.parse_postfix(progs[b]))
        else:
            a, c = pairs[b]
            assert O.sat(n, R, V, w, O.parse_postfix(progs[a])) != O.sat(n, R, V, w, O.parse_postfix(progs[c]))


# n, k, frames: several tiles of 4,096 frames with a ragged tail where the oracle finishes in seconds
SHAPES = [(6, 1, 9000), (6, 2, 700), (7, 0, 13000), (8, 1, 4500), (10, 1, 300), (12, 0, 8200),
          (13, 1, 40), (16, 0, 5000), (3, 2, 100), (1, 1, 5)]


@pytest.mark.parametrize("n,k,count", SHAPES)
def test_frame_list_parity(kb, vol, n, k, count):
    rel = F.stress_list(n, count)
    progs = formulas(1000 + n, 24, k)
    if k == 0:
        progs = progs + [W.to_postfix(W.alpha(m)) for m in (1, 2, 3)]
    code, offs = W.pack_programs(progs)
    want = vol.census_relations(code, offs, n, k, rel)
    h = kb.Programs(code, offs, k)
    succ = dev_succ(rel)
    got = kb.unpack(*kb.eval_frames(h, n, k, succ))
    same(got, want, f"sliced n={n} k={k}")
    certify(progs, got, n, k, rel)
    got_s = kb.unpack(*kb.eval_frames(h, n, k, succ, flags=kb.KERNEL_SCALAR))
    same(got_s, want, f"scalar n={n} k={k}")
    # pairs
    rng = np.random.Generator(np.random.PCG64(n))
    pairs = rng.integers(0, len(progs), size=(16, 2)).astype(np.uint32)
    pwant = vol.census_relations(code, offs, n, k, rel, pairs=pairs)
    pgot = kb.unpack(*kb.distinguish_pairs_frames(h, pairs, n, k, succ))
    same(pgot, pwant, f"pairs n={n} k={k}")
    certify(progs, pgot, n, k, rel, pairs=pairs)


def test_frame_list_deep_programs_and_chunks(kb, vol):
    """Programs that need more than four register-stack slots run on the scalar kernel inside the
    same call; chunked lists compose with KRIPKE_ACCUMULATE and index_base."""
    n, k = 7, 1
    rel = F.stress_list(n, 6000)
    deep = W.parse("((p & []p) | (<>p & [][]p)) -> (([]<>p | p) & (<>[]p -> (p & <><>p)))")
    progs = formulas(77, 10, k, budget=15, depth=6) + [W.to_postfix(deep)]
    code, offs = W.pack_programs(progs)
    want = vol.census_relations(code, offs, n, k, rel)
    h = kb.Programs(code, offs, k)
    succ = dev_succ(rel)
    got = kb.unpack(*kb.eval_frames(h, n, k, succ))
    same(got, want, "deep")
    c = w = None
    for a, b in [(0, 1000), (1000, 4100), (4100, 6000)]:
        part = succ[a * n:b * n].contiguous()
        flags = kb.ACCUMULATE if a else 0
        c, w = kb.eval_frames(h, n, k, part, index_base=a, flags=flags, counts_out=c, witness_out=w)
    same(kb.unpack(c, w), want, "chunked")


def test_frame_list_edges_and_errors(kb):
    import torch
    progs = [W.to_postfix(W.parse("[]p -> p")), W.to_postfix(W.parse("p -> p"))]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 1)
    empty = torch.zeros(0, dtype=torch.int16, device="cuda")
    got = kb.unpack(*kb.eval_frames(h, 6, 1, empty))
    assert got["models"].tolist() == [0, 0] and got["wit_f"].tolist() == [O.NO_WITNESS] * 2
    one = dev_succ(F.path(16)[None])
    with pytest.raises(kb.KripkeError) as e:
        kb.eval_frames(h, 17, 1, torch.zeros(17, dtype=torch.int16, device="cuda"))
    assert e.value.status == kb.EINVAL
    got = kb.unpack(*kb.eval_frames(h, 16, 1, one))          # n_vars * n = 16 <= 20 valuation bits
    assert int(got["frames"][0]) == 1 and int(got["models"][1]) == 0
    h2 = kb.Programs(code, offs, 2)
    with pytest.raises(kb.KripkeError) as e:
        kb.eval_frames(h2, 16, 2, one)                       # 32 valuation bits
    assert e.value.status == kb.EUNSUPPORTED
    with pytest.raises(kb.KripkeError) as e:
        kb.eval_frames(h, 6, 2, torch.zeros(12, dtype=torch.int16, device="cuda"))   # n_vars differs from the handle's
    assert e.value.status == kb.EINVAL


def test_in_library_generators_equal_the_numpy_restatement(kb, vol):
    """kripke_frames_generate (templates and seeded relations written on the device) against the
    counter-based generators of workloads/frames.py, mask by mask, for every generator and sizes 1..16; then a
    scan of a device-generated stress list against the oracle fed from the numpy side."""
    import torch
    for n in (1, 2, 3, 6, 9, 16):
        for gen in range(5):
            got = kb.frames_generate(gen, n, 777, 4242).cpu().numpy().view(np.uint16).reshape(777, n)
            want = F.succ_masks(F.generate_cb(gen, n, 777, 4242))
            assert (got == want).all(), (n, gen)
        for count in (3, 10, 11, 2050):
            got = kb.frames_generate(kb.GEN_STRESS, n, count, 99).cpu().numpy().view(np.uint16).reshape(count, n)
            assert (got == F.succ_masks(F.stress_list_cb(n, count, 99))).all(), (n, count)
    # the named templates are the paper's: the six-world path is Proposition 5's frame (2,4,8,16,32,0)
    t = kb.frames_generate(kb.GEN_TEMPLATES, 6, 10, 0).cpu().numpy().view(np.uint16).reshape(10, 6)
    assert t[0].tolist() == [2, 4, 8, 16, 32, 0]
    progs = [W.to_postfix(W.parse(s)) for s in ("[]p -> p", "[]p -> [][]p", "<>[]p -> []<>p", "[]<>[]<>T", "<>T")]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 1)
    n, count = 8, 5000
    succ = kb.frames_generate(kb.GEN_STRESS, n, count, 15437006)
    got = kb.unpack(*kb.eval_frames(h, n, 1, succ))
    want = vol.census_relations(code, offs, n, 1, F.stress_list_cb(n, count, 15437006))
    for key in ("models", "frames", "wit_f", "wit_v", "wit_w"):
        assert (got[key].astype(np.uint64) == want[key].astype(np.uint64)).all(), key
