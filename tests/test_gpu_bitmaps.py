"""Parity of the correspondence-recovery path (kripke_validity_bitmap, kripke_condition_bitmap,
kripke_match_bitmaps; Table 9 at P:366-376) with the oracle: bit-exact bitmaps.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

K, T, S4, S5 = 0, 1, 2, 3
AX = {name: W.to_postfix(t) for name, t in W.named_axioms().items()}
PAIRS = [("T", "reflexive"), ("4", "transitive"), ("B", "symmetric"), ("D", "serial"), ("5", "euclidean"),
         ("CD", "partially_functional"), ("C4", "dense"), ("G", "confluent")]


@pytest.fixture(scope="module")
def kb():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2606_15437_b200 import binding
    binding.load()
    return binding


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_condition_bitmaps_equal_the_oracle(kb, vol, n):
    total = 1 << (n * n)
    for name, cid in kb.COND.items():
        got = kb.bits_to_bool(kb.condition_bitmap(n, cid, K, 0, total), total)
        assert (got == vol.condition_bitmap(n, name).astype(bool)).all(), name
    # a class range with a ragged tail: reflexive frames, positions [5, 5 + count)
    tf = vol.class_frames(n, T)
    if len(tf) > 8:
        count = len(tf) - 7
        got = kb.bits_to_bool(kb.condition_bitmap(n, kb.COND["transitive"], T, 5, count), count)
        want = vol.condition_bitmap(n, "transitive").astype(bool)[tf[5:5 + count].astype(np.int64)]
        assert (got == want).all()


def test_n5_condition_counts(kb, vol):
    """Closed forms at n = 5: reflexive 2^20, symmetric 2^15, serial 31^5, partially
    functional 6^5, transitive 154,303 (OEIS A006905); the rest against the oracle's count."""
    total = 1 << 25
    want = {"reflexive": 1 << 20, "symmetric": 1 << 15, "serial": 31 ** 5, "partially_functional": 6 ** 5,
            "transitive": 154303}
    for name, cid in kb.COND.items():
        bm = kb.condition_bitmap(5, cid, K, 0, total).cpu().numpy().view(np.uint32)
        cnt = int(np.unpackbits(bm.view(np.uint8)).sum())
        assert cnt == want.get(name, vol.count_condition(5, name)), name


@pytest.mark.parametrize("n,cls", [(3, K), (4, K), (4, T), (4, S4), (4, S5), (2, K)])
def test_validity_bitmaps_equal_the_oracle(kb, vol, n, cls):
    progs = W.corpus_c2(300) + [AX[a] for a, _ in PAIRS] + [AX["K"], AX["M"]]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 2)
    size = kb.class_size(n, cls)
    for begin, count in ((0, size), (3, max(0, size - 10))):
        if count <= 0:
            continue
        got = kb.bits_to_bool(kb.validity_bitmap(h, n, 2, cls, begin, count), count)
        want = vol.validity(code, offs, n, 2, cls, begin, count).astype(bool)
        assert got.shape == want.shape and (got == want).all(), (n, cls, begin)
    # consistency with the census: valid frames = class size - refuting_frames
    full = kb.bits_to_bool(kb.validity_bitmap(h, n, 2, cls, 0, size), size)
    cen = kb.unpack(*kb.eval_batch_range(h, n, 2, cls, 0, size))
    assert (full.sum(axis=1) == size - cen["frames"].astype(np.int64)).all()


def test_table9_is_recovered_on_the_gpu(kb, vol):
    """Table 9: every Sahlqvist axiom's validity bitmap over all 65,536 four-world frames matches its
    own first-order correspondent in the library and no other; McKinsey's M matches none;
    K, p -> p match nothing in the library of proper conditions; corpus formulas that match a
    condition are re-checked against the oracle's bitmap of that condition."""
    import torch
    n, total = 4, 1 << 16
    names = list(kb.COND)
    lib = torch.stack([kb.condition_bitmap(n, kb.COND[c], K, 0, total) for c in names])
    progs = [AX[a] for a, _ in PAIRS] + [AX["M"], AX["K"], W.to_postfix(W.parse("p -> p"))] + W.corpus_c2(400)
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 2)
    bm = kb.validity_bitmap(h, n, 2, K, 0, total)
    match = kb.match_bitmaps(bm, lib).cpu().numpy()
    for i, (_, cond) in enumerate(PAIRS):
        assert match[i] == names.index(cond)
    assert match[8] == -1 and match[9] == -1 and match[10] == -1
    val = vol.validity(code, offs, n, 2)
    for b in np.nonzero(match >= 0)[0]:
        assert (val[b] == vol.condition_bitmap(n, names[match[b]])).all(), b
    for b in np.nonzero(match < 0)[0][:50]:
        assert not any((val[b] == vol.condition_bitmap(n, c)).all() for c in names), b


def test_bitmap_argument_errors(kb):
    h = kb.Programs(*W.pack_programs([AX["T"]]), 1)
    with pytest.raises(kb.KripkeError) as e:
        kb.validity_bitmap(h, 4, 1, K, 1 << 16, 1)
    assert e.value.status == kb.EINVAL
    with pytest.raises(kb.KripkeError) as e:
        kb.condition_bitmap(4, 8, K, 0, 16)
    assert e.value.status == kb.EINVAL
    assert kb.validity_bitmap(h, 4, 1, K, 0, 0).numel() == 0


@pytest.mark.parametrize("n,cond", [(4, "transitive"), (4, "confluent"), (3, "serial"), (5, "partially_functional")])
def test_frames_from_bitmap_is_the_extension(kb, vol, n, cond):
    """The compacted list holds exactly the frames whose bit is set (as successor masks, any order)."""
    total = 1 << (n * n)
    bm = kb.condition_bitmap(n, kb.COND[cond], K, 0, total)
    _, n_set = kb.frames_from_bitmap(n, K, 0, total, bm, 0)
    assert n_set == vol.count_condition(n, cond)
    succ, n2 = kb.frames_from_bitmap(n, K, 0, total, bm, n_set)
    assert n2 == n_set
    rows = succ.cpu().numpy().view(np.uint16).reshape(-1, n).astype(np.uint64)
    f = sum(rows[:, w] << np.uint64(w * n) for w in range(n))
    if n <= 4:
        want = np.nonzero(vol.condition_bitmap(n, cond))[0].astype(np.uint64)
    else:
        want = np.nonzero(kb.bits_to_bool(bm, total))[0].astype(np.uint64)
    assert (np.sort(f) == want).all()
    # a capacity smaller than the extension: only `capacity` frames are written, all of them members
    part, n3 = kb.frames_from_bitmap(n, K, 0, total, bm, 5)
    assert n3 == n_set and part.numel() == min(5, n_set) * n


def test_recovered_condition_reconfirmed_on_its_extension(kb, vol):
    """P:380 "each re-confirmed over all 33,554,432 five-world frames", composed from the bit-sliced
    kernels: T is refuted on no reflexive five-world frame (frame-list scan of the extension) and the
    census counts 2^25 - 2^20 refuting frames; 4 likewise on the 154,303 transitive frames."""
    total = 1 << 25
    for ax, cond, size in (("T", "reflexive", 1 << 20), ("4", "transitive", 154303)):
        bm = kb.condition_bitmap(5, kb.COND[cond], K, 0, total)
        succ, n_set = kb.frames_from_bitmap(5, K, 0, total, bm, size)
        assert n_set == size
        h = kb.Programs(*W.pack_programs([AX[ax], AX["B"]]), 1)
        on_ext = kb.unpack(*kb.eval_frames(h, 5, 1, succ))
        assert int(on_ext["frames"][0]) == 0 and int(on_ext["frames"][1]) > 0      # B fails on some of them
        cen = kb.unpack(*kb.eval_batch(h, 5, 1, K))
        assert int(cen["frames"][0]) == total - size


def test_k4_as_a_scan_class_by_composition(kb, vol):
    """Other frame classes (K4 = transitive frames, Table 4; serial, Euclidean, ...) need no kernel of
    their own: the condition's extension becomes a frame list and the frame-list scan runs on it.  K4 at
    n = 4: counts equal the oracle's census over the 3,994 transitive frames; the reported position maps
    back to a transitive frame that refutes."""
    n = 4
    total = 1 << (n * n)
    progs = W.corpus_c2(200) + [AX["4"], AX["T"], AX["K"]]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 2)
    bm = kb.condition_bitmap(n, kb.COND["transitive"], K, 0, total)
    succ, n_set = kb.frames_from_bitmap(n, K, 0, total, bm, 3994)
    assert n_set == 3994
    got = kb.unpack(*kb.eval_frames(h, n, 2, succ))
    frames = np.nonzero(vol.condition_bitmap(n, "transitive"))[0].astype(np.uint64)
    want = vol.census_list(code, offs, n, 2, frames)
    assert (got["models"] == want["models"]).all() and (got["frames"] == want["frames"]).all()
    assert int(got["frames"][200]) == 0 and int(got["frames"][201]) > 0 and int(got["models"][202]) == 0
    rows = succ.cpu().numpy().view(np.uint16).reshape(-1, n).astype(np.uint64)
    b = 201                                           # T is refuted on the non-reflexive transitive frames
    j = int(got["wit_f"][b])
    f = int(sum(int(rows[j, w]) << (w * n) for w in range(n)))
    assert f in set(int(x) for x in frames)
    from oracle import kripke_oracle as O
    assert O.check_witness(progs[b], n, 2, K, f, int(got["wit_v"][b]), int(got["wit_w"][b]))


def test_failure_density_panels_equal_the_oracle(kb, vol):
    """The atlas matrix: Atlas-3 = every K frame of 1..3 worlds; panels of explicit four- and
    five-world frames; a class range with a ragged size.  Counts of failing (valuation, world) pairs,
    bit-exact against the oracle."""
    import torch
    from workloads import frames as F
    progs = W.corpus_c2(250) + [AX[a] for a, _ in PAIRS]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 2)
    for n in (1, 2, 3):
        total = 1 << (n * n)
        got = kb.failure_density(h, n, 2, K, 0, total).cpu().numpy().view(np.uint32)
        assert (got == vol.failure_counts(code, offs, n, 2)).all(), n
    for n, count in ((4, 2048), (5, 1000), (8, 70)):
        rel = F.stress_list(n, count)
        k = 2 if n <= 5 else 1
        pr = progs if k == 2 else [W.to_postfix(W.parse(t)) for t in ("[]p -> p", "<>[]p", "[]<>[]p | p", "F")]
        c2, o2 = W.pack_programs(pr)
        hh = kb.Programs(c2, o2, k)
        succ = torch.from_numpy(F.succ_masks(rel).view(np.int16).reshape(-1).copy()).cuda()
        got = kb.failure_density_frames(hh, n, k, succ).cpu().numpy().view(np.uint32)
        assert (got == vol.failure_counts(c2, o2, n, k, rel=rel)).all(), n
    got = kb.failure_density(h, 4, 2, S4, 3, 300).cpu().numpy().view(np.uint32)
    assert (got == vol.failure_counts(code, offs, 4, 2, S4, 3, 300)).all()
    # zero density <=> valid frame (the validity bitmap of the same range)
    val = kb.bits_to_bool(kb.validity_bitmap(h, 4, 2, S4, 3, 300), 300)
    assert ((got == 0) == val).all()


def test_compiled_failure_density_equals_the_oracle(kb, vol):
    """kripke_failure_density over class ranges runs on the compiled bit-sliced kernels (a thread owns one
    frame and all its valuation words; without variables one frame per lane and the counts leave as three bit
    planes): every layout kind, every class, ragged ranges whose ends fall to the scalar kernel - bit-exact
    against the oracle's per-frame counts of failing (valuation, world) pairs."""
    k0 = W.pairs_c5(70)[0]
    k1 = [c for c in W.corpus_c4(600) if b"\x11" not in c and b"\x12" not in c][:50]
    k2 = W.corpus_c2(5624)[::47] + [AX[a] for a, _ in PAIRS]
    k3 = W.corpus_c4(60)
    cases = [(k2, 2, 3, K, 0, 512), (k2, 2, 4, K, 1000, 2048), (k2, 2, 5, K, (1 << 22) + 8, 4096),
             (k2, 2, 5, T, 77 * 4, 2048), (k2, 2, 5, S4, 0, 6940), (k2, 2, 4, S5, 0, 12), (k2, 2, 2, K, 0, 16),
             (k1, 1, 5, K, 4096, 8192), (k1, 1, 5, T, 0, 4096), (k1, 1, 6, K, 1 << 30, 1024), (k1, 1, 4, K, 0, 4096),
             (k0, 0, 5, K, 1024 * 3 + 4, 1024 * 5 + 8), (k0, 0, 4, K, 0, 1 << 16), (k0, 0, 5, T, 2048, 4096),
             (k0, 0, 6, K, (1 << 33) + 1024, 8192), (k0, 0, 3, K, 0, 512), (k0, 0, 5, S4, 0, 6940),
             (k3, 3, 4, K, 64, 256), (k3, 3, 5, K, 1 << 24, 16),
             # one frame per lane with a warp's words consecutive (units of 2^15 frames, rows staged through shared
             # memory and written 512 bytes per warp instruction): aligned units between two ragged ends; the same
             # programs in a one-variable batch (every count x 2^n)
             (k0, 0, 5, K, 3 * 32768 - 4000, 2 * 32768 + 8000), (k0, 0, 5, T, 32768 - 8, 2 * 32768 + 16),
             (k0, 0, 6, K, (1 << 35) - 32768, 3 * 32768), (k0[:20] + k1[:20], 1, 5, K, 5 * 32768 - 12, 32768 + 24)]
    for progs, k, n, cls, begin, count in cases:
        code, offs = W.pack_programs(progs)
        h = kb.Programs(code, offs, k)
        got = kb.failure_density(h, n, k, cls, begin, count).cpu().numpy().view(np.uint32)
        want = vol.failure_counts(code, offs, n, k, cls, begin, count)
        assert got.shape == want.shape and (got == want).all(), (k, n, cls, begin, count)
        info = h.last_run_info()
        if k * n >= 5 or (k == 0 and cls in (K, T) and n >= 3 and count >= 1024):
            assert info.kernel_family == 2, (k, n, cls)
    # an unaligned output row (count % 4 != 0) takes the scalar kernel and gives the same numbers
    code, offs = W.pack_programs(k2)
    h = kb.Programs(code, offs, 2)
    got = kb.failure_density(h, 4, 2, K, 5, 1001).cpu().numpy().view(np.uint32)
    assert (got == vol.failure_counts(code, offs, 4, 2, K, 5, 1001)).all() and h.last_run_info().kernel_family == 0
    # so does a range whose first frame is not a multiple of four (the rows' 16-byte chunks would be misaligned)
    code, offs = W.pack_programs(k0)
    h = kb.Programs(code, offs, 0)
    got = kb.failure_density(h, 5, 0, K, 32768 + 2, 32768).cpu().numpy().view(np.uint32)
    assert (got == vol.failure_counts(code, offs, 5, 0, K, 32768 + 2, 32768)).all() and h.last_run_info().kernel_family == 0
