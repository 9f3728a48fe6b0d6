"""Parity of the COMPILED bit-sliced scans (csrc/jit_*.cpp; the default engine) with the oracle run live,
for every layout kind the emitter has, and with the interpreted and scalar kernels; plus the boundary
conventions the compiled path touches (plan caching, streams, argument checks) and the multi-GPU exchange
step run on one device.  Bit-exact, no tolerance: everything is integer."""
import numpy as np
import pytest

import workloads as W
from oracle import kripke_oracle as O

pytestmark = pytest.mark.gpu

K, T, S4, S5 = 0, 1, 2, 3
KEYS = ("models", "frames", "wit_f", "wit_v", "wit_w")


@pytest.fixture(scope="module")
def kb():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2606_15437_b200 import binding
    binding.load()
    return binding


def same(got, want, what="", keys=KEYS):
    for key in keys:
        g, w = np.asarray(got[key]).astype(np.uint64), np.asarray(want[key]).astype(np.uint64)
        bad = np.nonzero(g != w)[0]
        assert len(bad) == 0, f"{what}: {key} differs at {bad[:5]}: got {g[bad[:5]]} want {w[bad[:5]]}"


def scan(kb, h, n, k, cls, begin, count, flags=0):
    return kb.unpack(*kb.eval_batch_range(h, n, k, cls, begin, count, flags))


ONE_VAR = None


def corpus(k):
    global ONE_VAR
    if k == 0:
        return W.pairs_c5(90)[0]
    if k == 1:
        if ONE_VAR is None:
            ONE_VAR = [c for c in W.corpus_c4(600) if b"\x11" not in c and b"\x12" not in c][:70]
        return ONE_VAR
    if k == 2:
        return W.corpus_c2(5624)[::19] + [W.to_postfix(t) for t in W.named_axioms().values()]
    return W.corpus_c4(140)


# (n, k, class, begin, count): windows that hold whole scan units of every variable-count group of the shape
# plus ragged ends on both sides (the ends run on the scalar kernel), or full small classes
SHAPES = [
    (5, 2, K, 1024 * 31 - 3, 2100), (5, 2, T, 1024 * 7 - 5, 2100), (5, 2, S4, 100, 3000), (5, 2, S5, 0, 52),
    (5, 1, K, 1024 * 5 - 1, 3000), (5, 1, T, 77, 2500), (5, 1, S4, 0, 6942),
    (5, 0, K, 1024 * 9 - 7, 4100), (5, 0, T, 1000, 3000),
    (4, 2, K, 0, 1 << 16), (4, 2, T, 0, 1 << 12), (4, 2, S4, 0, 355), (4, 2, S5, 0, 15),
    (4, 1, K, 5, 40000), (4, 0, K, 0, 1 << 16), (4, 3, K, 1000, 700), (4, 3, S4, 0, 355),
    (3, 2, K, 0, 512), (3, 2, T, 0, 64), (3, 1, K, 0, 512), (3, 0, K, 0, 512), (3, 3, S4, 0, 29),
    (2, 2, K, 0, 16), (2, 1, T, 0, 4),
    (6, 0, K, (1 << 30) - 5000, 12000), (6, 1, K, (1 << 33) + 11, 4100), (6, 2, K, (1 << 35) - 40, 300),
    (5, 3, K, (1 << 24) + 3, 40), (5, 3, T, 12345, 40),
]


@pytest.mark.parametrize("n,k,cls,begin,count", SHAPES)
def test_compiled_scan_equals_oracle(kb, vol, n, k, cls, begin, count):
    progs = corpus(k)
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, k)
    want = vol.census(code, offs, n, k, cls, begin, count)
    got = scan(kb, h, n, k, cls, begin, count)
    info = h.last_run_info()
    same(got, want, f"compiled n={n} k={k} cls={cls} [{begin},+{count})")
    layout = kb.debug_jit_source(code, offs, k, n, cls, k) is not None
    if layout and count >= 2048:
        assert info.kernel_family == 2 and info.jit_programs > 0 and info.jit_compile_seconds >= 0.0
    # the ablation modes give the same records
    same(scan(kb, h, n, k, cls, begin, count, kb.NO_SUBTERM_SHARING), want, "no subterm sharing")
    if len(progs) <= 150:
        same(scan(kb, h, n, k, cls, begin, count, kb.NO_SHARING | kb.FULL_SWEEP), want, "no sharing, full sweep")
    # certificates (Definition 1) for a sample
    for b in range(0, len(progs), 7):
        f = int(got["wit_f"][b])
        if f != O.NO_WITNESS:
            assert O.check_witness(progs[b], n, k, cls, f, int(got["wit_v"][b]), int(got["wit_w"][b]))


def test_compiled_equals_interpreted_and_scalar_on_c2(kb):
    """The three kernel families on all of C2 (n=4, four classes) and on an n=5 window."""
    progs = W.corpus_c2()
    h = kb.Programs(*W.pack_programs(progs), 2)
    for n, cls, begin, count in ((4, K, 0, 1 << 16), (4, T, 0, 1 << 12), (4, S4, 0, 355), (5, K, 3 << 20, 1 << 13),
                                 (5, T, 1 << 19, 1 << 12), (5, S4, 0, 6942)):
        a = scan(kb, h, n, 2, cls, begin, count, kb.KERNEL_JIT)
        assert h.last_run_info().kernel_family == 2
        b = scan(kb, h, n, 2, cls, begin, count, kb.KERNEL_SLICED)
        assert h.last_run_info().kernel_family == 1
        same(a, b, f"compiled vs interpreted n={n} cls={cls}")
        if n == 4:
            same(a, scan(kb, h, n, 2, cls, begin, count, kb.KERNEL_SCALAR), f"compiled vs scalar n={n} cls={cls}")


def test_rewrites_and_plan_cache_give_the_same_records(kb, vol):
    """The guarded-root and box-distribution rewrites (on by default) leave every record unchanged: default =
    each ablation flag = the oracle, on windows of K and T at n = 5 and on all of S4; a second handle over the same
    bytes takes its plan from the process-wide cache (nothing is compiled) and gives the same records."""
    extra = ["[]p", "[][]p", "[](p & q)", "[]p & []q", "[][](p -> q) & p", "[]F", "[][]F", "[]([]p & q)",
             "[]([]F | p)", "[]p & ([]q & ~[](p & q))", "[](p & []q) -> [](q & []p)", "[](p & q & []p)", "[][][]q"]
    progs = W.corpus_c2(5624)[::13] + [W.to_postfix(W.parse(t)) for t in extra]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 2)
    for cls, begin, count in ((K, 1024 * 77, 2048), (T, 1024 * 3, 2048), (S4, 0, 6942)):
        want = vol.census(code, offs, 5, 2, cls, begin, count)
        same(scan(kb, h, 5, 2, cls, begin, count), want, f"default cls={cls}")
        assert h.last_run_info().kernel_family == 2
        ops = h.last_run_info().logic_instr_per_frame
        for fl in (kb.NO_GUARDED_ROOTS, kb.NO_BOX_DISTRIBUTION, kb.NO_GUARDED_ROOTS | kb.NO_BOX_DISTRIBUTION):
            same(scan(kb, h, 5, 2, cls, begin, count, fl), want, f"flags={fl} cls={cls}")
        assert h.last_run_info().logic_instr_per_frame > ops          # the rewrites do remove work
    h2 = kb.Programs(code, offs, 2)
    got = scan(kb, h2, 5, 2, K, 1024 * 77, 2048)
    assert h2.last_run_info().jit_compile_seconds == 0.0
    same(got, vol.census(code, offs, 5, 2, K, 1024 * 77, 2048), "plan from the cache")


def test_compiled_pairs_equal_oracle(kb, vol):
    progs, pairs, _ = W.pairs_c5(400)
    pairs = np.array(pairs, np.uint32)
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 0)
    for n, begin, count in ((4, 0, 1 << 16), (5, (1 << 20) - 3, 5000), (6, 17335328 - 3000, 6000)):
        want = vol.census(code, offs, n, 0, K, begin, count, pairs=pairs)
        got = kb.unpack(*kb.distinguish_pairs(h, pairs, n, 0, K, begin, count))
        same(got, want, f"pairs n={n}")
        assert h.last_run_info().kernel_family == 2
    # pairs with variables (k = 2): the witness valuation is lexicographically first
    p2 = W.corpus_c2(200)
    pr2 = np.array([[i, i + 1] for i in range(0, 198, 2)], np.uint32)
    c2, o2 = W.pack_programs(p2)
    h2 = kb.Programs(c2, o2, 2)
    for n, cls, begin, count in ((4, K, 0, 1 << 16), (5, T, 4000, 2100)):
        want = vol.census(c2, o2, n, 2, cls, begin, count, pairs=pr2)
        same(kb.unpack(*kb.distinguish_pairs(h2, pr2, n, 2, cls, begin, count)), want, f"k=2 pairs n={n}")


def test_forced_compiled_needs_an_aligned_range(kb):
    import torch
    progs = W.corpus_c2(64)
    h = kb.Programs(*W.pack_programs(progs), 2)
    c = torch.zeros((64, 2), dtype=torch.int64, device="cuda")
    w = torch.zeros((64, 2), dtype=torch.int64, device="cuda")
    lib = kb.load()
    # one-variable programs are scanned 32 frames per unit: a range that is not a multiple cannot be forced
    rc = lib.kripke_eval_batch_range(h._h, 5, 2, K, 3, 1000, kb.KERNEL_JIT, c.data_ptr(), w.data_ptr(), None)
    assert rc == kb.EUNSUPPORTED
    rc = lib.kripke_eval_batch_range(h._h, 5, 2, K, 1024, 2048, kb.KERNEL_JIT, c.data_ptr(), w.data_ptr(), None)
    assert rc == kb.OK
    rc = lib.kripke_eval_batch_range(h._h, 2, 2, K, 0, 16, kb.KERNEL_JIT | kb.FULL_SWEEP, c.data_ptr(), w.data_ptr(), None)
    assert rc == kb.OK                                    # n=2, k=2: 16 frames x 16 valuations = 8 words
    h0 = kb.Programs(*W.pack_programs(W.pairs_c5(4)[0]), 0)
    c0 = torch.zeros((len(W.pairs_c5(4)[0]), 2), dtype=torch.int64, device="cuda")
    rc = lib.kripke_eval_batch_range(h0._h, 2, 0, K, 0, 16, kb.KERNEL_JIT, c0.data_ptr(), c0.clone().data_ptr(), None)
    assert rc == kb.EUNSUPPORTED                          # 16 models: no compiled layout


def test_bad_arguments_leave_no_plan_behind(kb, vol):
    """a call with the wrong n_vars must fail before a plan is built or cached; the next valid
    call must scan every record (n=6, k=3 vs k=4 used to share a cache key)."""
    import torch
    progs = [c for c in W.corpus_c4(200)][:24]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 3)
    c = torch.zeros((24, 2), dtype=torch.int64, device="cuda")
    w = torch.zeros((24, 2), dtype=torch.int64, device="cuda")
    lib = kb.load()
    for bad_k in (4, 2, 0):
        rc = lib.kripke_eval_batch_range(h._h, 4, bad_k, K, 0, 64, 0, c.data_ptr(), w.data_ptr(), None)
        assert rc == kb.EINVAL
    rc = lib.kripke_eval_batch_range(h._h, 4, 3, 7, 0, 64, 0, c.data_ptr(), w.data_ptr(), None)
    assert rc == kb.EINVAL
    rc = lib.kripke_eval_batch_range(h._h, 4, 3, K, 0, 64, 1 << 20, c.data_ptr(), w.data_ptr(), None)
    assert rc == kb.EINVAL
    got = scan(kb, h, 4, 3, K, 0, 4096)
    same(got, vol.census(code, offs, 4, 3, K, 0, 4096), "after rejected calls")


def test_pair_scans_on_two_streams_and_plan_reuse(kb, vol):
    """kripke_distinguish_pairs enqueues and returns: two pair scans of one handle issued back to back on
    two streams (the second waits on the device for the first; the host never blocks), then the same lists
    again (cached plans: no new compilation)."""
    import torch
    progs, pairs, _ = W.pairs_c5(300)
    pairs = np.array(pairs, np.uint32)
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 0)
    pa, pb = pairs[:150], pairs[150:320]
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    kb.distinguish_pairs(h, pa, 5, 0, K, 0, 1 << 20)              # builds plan a
    kb.distinguish_pairs(h, pb, 5, 0, K, 0, 1 << 20)              # builds plan b
    torch.cuda.synchronize()
    ra = kb.distinguish_pairs(h, pa, 5, 0, K, 1 << 20, 1 << 22, stream=s1)
    assert h.last_run_info().jit_compile_seconds >= 0.0
    rb = kb.distinguish_pairs(h, pb, 5, 0, K, 1 << 20, 1 << 22, stream=s2)
    ra2 = kb.distinguish_pairs(h, pa, 5, 0, K, 1 << 20, 1 << 22, stream=s1)
    torch.cuda.synchronize()
    wa = vol.census(code, offs, 5, 0, K, 1 << 20, 1 << 12, pairs=pa)          # oracle on a prefix of the range
    ga = kb.unpack(*kb.distinguish_pairs(h, pa, 5, 0, K, 1 << 20, 1 << 12))
    same(ga, wa, "pairs a, prefix")
    same(kb.unpack(*ra), kb.unpack(*ra2), "same list twice")
    # against one scan on the default stream
    same(kb.unpack(*rb), kb.unpack(*kb.distinguish_pairs(h, pb, 5, 0, K, 1 << 20, 1 << 22)), "pairs b")
    same(kb.unpack(*ra), kb.unpack(*kb.distinguish_pairs(h, pa, 5, 0, K, 1 << 20, 1 << 22)), "pairs a")


def test_exchange_step_on_one_device(kb, vol):
    """the multi-GPU combine - counts by SUM, witnesses by MIN of 64-bit keys - run on one device:
    two half ranges of each class scanned into separate buffers, kripke_witness_to_keys on each, minimum /
    sum, kripke_keys_to_witness; equal to the full scan and to the oracle.  The batch has a record with no
    witness at all (the K axiom) and records whose first countermodel lies in the second half."""
    import torch
    progs = W.corpus_c2(300) + [W.to_postfix(W.named_axioms()["K"]), W.to_postfix(W.parse("p -> p"))]
    # valid on the first frame of the class (K: no edge at all; T: only the loops), refuted on later ones
    progs += [W.to_postfix(W.parse(t)) for t in ("[]F", "p -> []p", "<>p -> p", "[][]F")]
    code, offs = W.pack_programs(progs)
    h = kb.Programs(code, offs, 2)
    for n, cls in ((4, K), (4, T), (4, S4), (4, S5), (5, S4)):
        total = kb.class_size(n, cls)
        full = kb.unpack(*kb.eval_batch_range(h, n, 2, cls, 0, total))
        want = vol.census(code, offs, n, 2, cls)
        same(full, want, f"full scan n={n} cls={cls}")
        for cut in (1, total // 2 + 3):
            parts = []
            for a, b in ((0, cut), (cut, total)):
                c, w = kb.eval_batch_range(h, n, 2, cls, a, b - a)
                parts.append((c.clone(), kb.witness_to_keys(w, n, 2).clone()))
            counts = parts[0][0] + parts[1][0]
            keys = torch.minimum(parts[0][1], parts[1][1])
            got = kb.unpack(counts, kb.keys_to_witness(keys, n, 2))
            same(got, want, f"combined ranges n={n} cls={cls} cut={cut}")
            assert int(got["wit_f"][300]) == O.NO_WITNESS and int(got["models"][300]) == 0
            first = kb.unpack(parts[0][0], kb.keys_to_witness(parts[0][1], n, 2))
            second = np.nonzero((first["wit_f"] == O.NO_WITNESS) & (got["wit_f"] != O.NO_WITNESS))[0]
            if cut == 1:
                assert len(second) >= 3, "records whose least (f, v) lies in the second range"


def test_cache_clear_recompiles_and_gives_the_same_records(kb):
    """kripke_jit_cache_clear: refused while a handle exists (its plans hold kernels of the cached modules);
    with none alive it unloads the modules, and the next scan of the same batch compiles again and returns the
    same records."""
    import gc
    import torch
    gc.collect()
    progs = corpus(2)[:60]
    h = kb.Programs(*W.pack_programs(progs), 2)
    before = scan(kb, h, 4, 2, K, 0, 1 << 16)
    assert h.last_run_info().kernel_family == 2
    with pytest.raises(kb.KripkeError) as err:
        kb.jit_cache_clear()
    assert err.value.status == kb.EINVAL
    h.destroy()
    assert kb.jit_cache_clear() >= 1                 # at least this batch's module was loaded
    assert kb.jit_cache_clear() == 0                 # nothing left
    h = kb.Programs(*W.pack_programs(progs), 2)
    after = scan(kb, h, 4, 2, K, 0, 1 << 16)
    assert h.last_run_info().jit_compile_seconds > 0  # rebuilt, not found in a cache
    same(after, before, "after a cache clear")
    again = scan(kb, h, 4, 2, K, 0, 1 << 16)
    torch.cuda.synchronize()
    same(again, before, "second scan on the rebuilt plan")
    h.destroy()


def test_two_handles_on_two_streams_and_a_refused_call_in_between(kb, vol):
    """Two handles scan on their own streams; one is destroyed while the other still has work queued (destroy
    waits for the handle's own last scan only); a forced-family call that is refused (unaligned range for the
    compiled kernels) sits between two good scans of the same handle on different streams and must not disturb
    either.  Every record equals the oracle's."""
    import torch
    progs_a, progs_b = corpus(2)[:120], corpus(1)[:40]
    code_a, offs_a = W.pack_programs(progs_a)
    code_b, offs_b = W.pack_programs(progs_b)
    want_a = vol.census(code_a, offs_a, 4, 2, K, 1 << 12, 1 << 13)
    want_a2 = vol.census(code_a, offs_a, 4, 2, K, 3, 1000)
    want_b = vol.census(code_b, offs_b, 4, 1, T, 0, 1 << 12)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    ha, hb = kb.Programs(code_a, offs_a, 2), kb.Programs(code_b, offs_b, 1)
    ca, wa = kb.eval_batch_range(ha, 4, 2, K, 1 << 12, 1 << 13, 0, stream=s1)
    cb, wb = kb.eval_batch_range(hb, 4, 1, T, 0, 1 << 12, 0, stream=s2)
    with pytest.raises(kb.KripkeError) as err:                       # 3 is not a multiple of the scan unit
        kb.eval_batch_range(ha, 4, 2, K, 3, 1000, kb.KERNEL_JIT, stream=s2)
    assert err.value.status == kb.EUNSUPPORTED
    hb.destroy()                                                     # ha's scan on s1 may still be running
    torch.cuda.synchronize()
    got_a, got_b = kb.unpack(ca, wa), kb.unpack(cb, wb)
    ca2, wa2 = kb.eval_batch_range(ha, 4, 2, K, 3, 1000, 0, stream=s2)   # same handle, other stream, ragged range
    torch.cuda.synchronize()
    same(got_a, want_a, "handle a, stream 1")
    same(got_b, want_b, "handle b, stream 2")
    same(kb.unpack(ca2, wa2), want_a2, "handle a again on stream 2 after the refused call")
    ha.destroy()
