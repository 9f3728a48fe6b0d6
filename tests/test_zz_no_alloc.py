"""kripke_eval_batch_static - the scan for callers that cannot allocate device memory.

Some users of the library cannot call cudaMalloc: their process's device memory is owned by another
allocator (a torch caching allocator that was given the card, a server's pre-reserved pool), or they
run next to streams that cudaMalloc / cudaFree's device-wide synchronisation would stall.  For them the
library has one entry point whose working memory is a fixed block inside the library image instead of a
handle's allocations.  These tests check that it returns exactly what the handle path returns (integer
results: bit for bit, the tolerance of every parity test here), including when calls follow each other
and the second finds the first one's leftovers in the shared block.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should
not hide the parity tests.  Nothing in it depends on what ran before it in the process.
"""
import numpy as np
import pytest

import workloads as W

K, T, S4, S5 = 0, 1, 2, 3
KEYS = ("models", "frames", "wit_f", "wit_v", "wit_w")


@pytest.fixture(scope="module")
def kb():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2606_15437_b200 import binding
    binding.load()
    return binding


def outputs(n, fill):
    """The caller's own output tensors, pre-filled with junk the call has to overwrite."""
    import torch
    return (torch.full((n, 2), fill, dtype=torch.int64, device="cuda"),
            torch.full((n, 2), fill, dtype=torch.int64, device="cuda"))


def static_scan(kb, progs, n, k, cls, begin, count, flags=0, out=None, fill=-7):
    code, offsets = W.pack_programs(progs)
    c, w = out if out is not None else outputs(len(progs), fill)
    kb.eval_batch_static(code, offsets, n, k, cls, begin, count, c, w, flags)
    return kb.unpack(c, w)


def handle_scan(kb, progs, n, k, cls, begin, count, flags=0):
    h = kb.Programs(*W.pack_programs(progs), k)
    res = kb.unpack(*kb.eval_batch_range(h, n, k, cls, begin, count, flags))
    h.destroy()
    return res


def same(got, want, what):
    for key in KEYS:
        g, w = np.asarray(got[key]).astype(np.uint64), np.asarray(want[key]).astype(np.uint64)
        bad = np.nonzero(g != w)[0]
        assert len(bad) == 0, f"{what}: {key} differs at {bad[:5]}: got {g[bad[:5]]} want {w[bad[:5]]}"


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_handle_path(kb):
    """Two different scans back to back on one stream.  The second is smaller than the first (fewer
    formulas, shorter code, a class that needs the table section), so every accumulator, offset and code
    byte it does not overwrite still holds the first scan's values: a missing re-initialisation shows as a
    count that is too large or a witness that belongs to the other batch.  Then the first scan again, to
    see that the second left nothing behind either."""
    import torch
    first = W.corpus_c2(700)                       # 700 formulas over {p, q}: class K, n = 3, ragged range
    second = W.corpus_c1(90)                       # 90 formulas: class S4 on four worlds (355 preorders)
    a = static_scan(kb, first, 3, 2, K, 5, 500)
    b = static_scan(kb, second, 4, 2, S4, 0, kb.class_size(4, S4), fill=-1)
    a2 = static_scan(kb, first, 3, 2, K, 5, 500, fill=0)
    torch.cuda.synchronize()
    want_a = handle_scan(kb, first, 3, 2, K, 5, 500)                       # the default (compiled) engine
    want_b = handle_scan(kb, second, 4, 2, S4, 0, kb.class_size(4, S4))
    same(a, want_a, "first call")
    same(b, want_b, "second call")
    same(a2, want_a, "first scan repeated after the second")
    same(a, handle_scan(kb, first, 3, 2, K, 5, 500, kb.KERNEL_SCALAR), "first call vs the scalar kernel on a handle")
    assert int(a["models"].sum()) > 0 and int(b["models"].sum()) > 0      # the comparison is not over zeros


@pytest.mark.gpu
def test_classes_chunks_and_reduce_modes(kb):
    """Every class, a range cut into chunks that are added up with KRIPKE_ACCUMULATE into the same output
    tensors, and the three reduction modes - each equal to one handle-path scan of the whole range."""
    progs = W.corpus_c2(160)
    for cls, n in ((K, 4), (T, 4), (S4, 5), (S5, 5)):
        size = kb.class_size(n, cls)
        count = min(size, 3000)
        want = handle_scan(kb, progs, n, 2, cls, 0, count)
        out = outputs(len(progs), 123)
        cuts = [0, count // 3 + 1, count // 2, count]
        for i in range(3):
            got = static_scan(kb, progs, n, 2, cls, cuts[i], cuts[i + 1] - cuts[i],
                              flags=kb.ACCUMULATE if i else 0, out=out)
        same(got, want, f"class {cls} in three chunks")
    for mode in (kb.REDUCE_BLOCK, kb.REDUCE_WARP, kb.REDUCE_THREAD):
        same(static_scan(kb, progs, 3, 2, K, 0, 512, flags=mode), handle_scan(kb, progs, 3, 2, K, 0, 512),
             f"reduce mode {mode >> 8}")
    # an empty range: zero counts, no witness
    empty = static_scan(kb, progs, 3, 2, K, 17, 0)
    assert not empty["models"].any() and not empty["frames"].any() and (empty["wit_f"] == kb.NO_WITNESS).all()


@pytest.mark.gpu
def test_the_call_allocates_no_device_memory(kb):
    """Free device memory as the driver reports it is the same before and after (the output tensors exist
    before the first reading, and the first call's set-up is behind us)."""
    import torch
    progs = W.corpus_c2(64)
    out = outputs(len(progs), 0)
    static_scan(kb, progs, 3, 2, K, 0, 512, out=out)
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        static_scan(kb, progs, 3, 2, K, 0, 512, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= before


def test_sizes_beyond_the_static_block_are_refused():
    """Host-side checks come before any CUDA call, so this runs without a GPU: a batch larger than
    KRIPKE_STATIC_MAX_FORMULAS, a class table larger than KRIPKE_STATIC_MAX_CLASS_FRAMES and flags the
    entry point does not take are rejected with the documented status; the limits in the binding are the
    header's."""
    import ctypes
    import os
    import re
    from paper_2606_15437_b200 import binding as kb
    lib = kb.load()
    header = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "kripke.h")).read()
    for name in ("STATIC_MAX_FORMULAS", "STATIC_MAX_CLASS_FRAMES", "STATIC_SCRATCH_BYTES"):
        assert int(re.search(rf"#define KRIPKE_{name} (\d+)u", header).group(1)) == getattr(kb, name)

    def call(progs, n, k, cls, begin, count, flags=0, out=0x1000):
        code, offsets = kb._host(*W.pack_programs(progs))
        return lib.kripke_eval_batch_static(code.ctypes.data, offsets.ctypes.data, len(progs), n, k, cls, begin, count,
                                            flags, ctypes.c_void_p(out), ctypes.c_void_p(out), None)

    top = bytes([0x00])
    assert call([top] * (kb.STATIC_MAX_FORMULAS + 1), 3, 1, K, 0, 1) == kb.EUNSUPPORTED
    assert call([top], 6, 1, S4, 0, 1) == kb.EUNSUPPORTED               # 209,527 preorders on six worlds
    assert call([top], 3, 1, K, 0, 1, flags=kb.KERNEL_JIT) == kb.EINVAL
    assert call([top], 3, 1, K, 500, 100) == kb.EINVAL                  # range outside the 512 frames
    assert call([bytes([0x30])], 3, 1, K, 0, 1) == kb.EPROGRAM          # "and" with an empty stack
    assert call([top], 3, 1, K, 0, 1, out=0) == kb.EINVAL               # no output arrays
