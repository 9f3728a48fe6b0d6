"""Seeded fuzz parity of the default (compiled) engine against the oracle run live: random batches of random
formulas (different sizes, depths, atom sets - duplicates, constants, complemented and permuted variants
included on purpose), random shapes and frame windows with ragged ends, single formulas, pairs and failure
densities.  Everything the rewrites touch (guarded roots, box distribution, canonical variable order and
polarity, the nested valuation loop, packed counters, kernel splitting) is on.  Bit-exact, no tolerance."""
import numpy as np
import pytest

import workloads as W
from oracle import kripke_oracle as O

pytestmark = pytest.mark.gpu

KEYS = ("models", "frames", "wit_f", "wit_v", "wit_w")
VARS = "pqrs"


@pytest.fixture(scope="module")
def kb():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2606_15437_b200 import binding
    binding.load()
    return binding


def _batch(rng, k, count):
    """Random formulas over the first k variables and the constants, plus variants of some of them with the
    variables permuted / complemented and with redundant double negations."""
    atoms = VARS[:k] + "TF" if rng.below(3) else (VARS[:k] or "TF")
    out = []
    while len(out) < count:
        t = W.gen_formula(rng, 3 + rng.below(12), 1 + rng.below(5), atoms)
        out.append(t)
        if k and rng.below(4) == 0:
            perm = list(range(k))
            for i in range(k - 1, 0, -1):
                j = rng.below(i + 1)
                perm[i], perm[j] = perm[j], perm[i]
            mask = rng.below(1 << k)

            def vary(u):
                if u[0] == "var":
                    v = ("var", perm[u[1]])
                    return ("not", v) if (mask >> u[1]) & 1 else v
                return (u[0],) + tuple(vary(c) for c in u[1:])
            out.append(vary(t))
        if rng.below(8) == 0:
            out.append(("not", ("not", t)))
    return [W.to_postfix(t) for t in out[:count]]


def _window(rng, total, width):
    width = min(width, total)
    begin = rng.below(total - width + 1)
    return begin, width


@pytest.mark.parametrize("seed", [15437101 + i for i in range(10)])
def test_fuzz_single_formulas(kb, vol, seed):
    rng = W.SplitMix64(seed)
    for _ in range(10):
        k = rng.below(4)
        n = 2 + rng.below(4) if k < 3 else 2 + rng.below(3)            # n <= 5 (k = 3: n <= 4): the oracle finishes in seconds
        cls = rng.below(4)
        progs = _batch(rng, k, 20 + rng.below(120))
        code, offs = W.pack_programs(progs)
        total = kb.class_size(n, cls)
        width = (3000 >> (k * max(n - 3, 0))) + rng.below(2000 >> (k * max(n - 3, 0)) or 1) + 1
        begin, count = _window(rng, total, max(width, 40))
        h = kb.Programs(code, offs, k)
        got = kb.unpack(*kb.eval_batch_range(h, n, k, cls, begin, count))
        want = vol.census(code, offs, n, k, cls, begin, count)
        for key in KEYS:
            g, w = got[key].astype(np.uint64), want[key].astype(np.uint64)
            bad = np.nonzero(g != w)[0]
            assert len(bad) == 0, (seed, n, k, cls, begin, count, key, bad[:5], g[bad[:5]], w[bad[:5]],
                                   [W.to_text(W.from_postfix(progs[b])) for b in bad[:3]])
        for b in range(0, len(progs), 11):
            if int(got["wit_f"][b]) != O.NO_WITNESS:
                assert O.check_witness(progs[b], n, k, cls, int(got["wit_f"][b]), int(got["wit_v"][b]), int(got["wit_w"][b]))
        h.destroy()


@pytest.mark.parametrize("seed", [15437201 + i for i in range(6)])
def test_fuzz_pairs_and_densities(kb, vol, seed):
    rng = W.SplitMix64(seed)
    for _ in range(6):
        k = rng.below(3)
        n = 3 + rng.below(3) if k < 2 else 3 + rng.below(2)
        cls = rng.below(4)
        progs = _batch(rng, k, 40 + rng.below(60))
        code, offs = W.pack_programs(progs)
        P = 30 + rng.below(40)
        pairs = np.array([[rng.below(len(progs)), rng.below(len(progs))] for _ in range(P)], np.uint32)
        total = kb.class_size(n, cls)
        begin, count = _window(rng, total, 600 + rng.below(1500))
        h = kb.Programs(code, offs, k)
        got = kb.unpack(*kb.distinguish_pairs(h, pairs, n, k, cls, begin, count))
        want = vol.census(code, offs, n, k, cls, begin, count, pairs=pairs)
        for key in KEYS:
            assert (got[key].astype(np.uint64) == want[key].astype(np.uint64)).all(), (seed, "pairs", n, k, cls, begin, count, key)
        # failure densities on a window whose start is a multiple of four (compiled kernels) and on a ragged one
        for b0, cnt in ((begin & ~3, min(count & ~3, total - (begin & ~3)) & ~3), (begin, min(count, 257))):
            if cnt <= 0 or k * n > 20:
                continue
            d = kb.failure_density(h, n, k, cls, b0, cnt).cpu().numpy().astype(np.uint64)
            dw = vol.failure_counts(code, offs, n, k, cls, b0, cnt).astype(np.uint64).reshape(len(progs), -1)
            assert (d == dw).all(), (seed, "density", n, k, cls, b0, cnt)
        h.destroy()
