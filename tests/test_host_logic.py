"""Host-side logic of libkripke_b200.so, testable without a GPU: the ABI surface, the program
validator, the lowering to micro-ops and the class-table enumerator.  No compute call is made."""
import ctypes
import os
import re

import numpy as np
import pytest

import workloads as W
from paper_2606_15437_b200 import binding as kb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "kripke.h")).read()
    declared = set(re.findall(r"^(?:int|const char \*)\s*(kripke_[a-z0-9_]+)\(", header, re.M))
    assert declared == set(kb.EXPORTS)
    lib = kb.load()
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.kripke_version()


def _validate(progs, n_vars):
    code, offs = W.pack_programs(progs)
    return kb.validate_programs(code, offs, n_vars)


def test_validator_accepts_corpora_and_reports_depth():
    assert _validate(W.corpus_c1(200), 2) <= 4
    assert _validate(W.corpus_c4(200), 3) <= 8
    assert _validate([W.to_postfix(W.parse("p&(q&(p&(q&p)))"))], 2) == 5


@pytest.mark.parametrize("prog,nvars,status", [
    (bytes([0x10, 0x30]), 2, kb.EPROGRAM),            # binary operator underflow
    (bytes([0x20]), 2, kb.EPROGRAM),                  # unary operator underflow
    (bytes([0x10, 0x11]), 2, kb.EPROGRAM),            # leaves two values
    (bytes([0x10, 0x7f]), 2, kb.EPROGRAM),            # bad opcode
    (bytes([0x12]), 2, kb.EPROGRAM),                  # variable index >= n_vars
    (b"", 2, kb.EPROGRAM),                            # empty program
    (bytes([0x10] * 17 + [0x30] * 16), 1, kb.EUNSUPPORTED),   # needs 17 stack slots
    (bytes([0x10] + [0x20] * 64), 1, kb.EUNSUPPORTED),        # longer than 64 opcodes
])
def test_validator_rejects(prog, nvars, status):
    with pytest.raises(kb.KripkeError) as e:
        _validate([prog], nvars)
    assert e.value.status == status


def test_validator_argument_errors():
    lib = kb.load()
    assert lib.kripke_validate_programs(None, None, 0, 2, None) == kb.EINVAL
    offs = np.array([0, 1], np.uint32)
    assert lib.kripke_validate_programs(None, offs.ctypes.data, 1, 2, None) == kb.EINVAL
    code = np.array([0x10], np.uint8)
    assert lib.kripke_validate_programs(code.ctypes.data, offs.ctypes.data, 1, 5, None) == kb.EINVAL
    bad = np.array([1, 0], np.uint32)
    assert lib.kripke_validate_programs(code.ctypes.data, bad.ctypes.data, 1, 2, None) == kb.EINVAL


def test_class_sizes():
    pre = [1, 4, 29, 355, 6942, 209527]       # OEIS A000798
    bell = [1, 2, 5, 15, 52, 203]            # OEIS A000110
    for n in range(1, 7):
        assert kb.class_size(n, kb.CLASS_K) == 1 << (n * n)
        assert kb.class_size(n, kb.CLASS_T) == 1 << (n * n - n)
        assert kb.class_size(n, kb.CLASS_S4) == pre[n - 1]
        assert kb.class_size(n, kb.CLASS_S5) == bell[n - 1]
    with pytest.raises(kb.KripkeError):
        kb.class_size(7, 0)
    with pytest.raises(kb.KripkeError):
        kb.class_size(3, 4)


# --- a tiny interpreter of the micro-ops on ONE model (n-bit masks), test-side only --------------
def _run_ucode(uc, n, succ, vals):
    full = (1 << n) - 1
    D = [0, 0, 0, 0]

    def box(x):
        return sum(1 << w for w in range(n) if succ[w] & ~x & full == 0)

    def dia(x):
        return sum(1 << w for w in range(n) if succ[w] & x)

    leaves = {0: vals[0], 1: box(0), 2: box(vals[0]), 3: dia(vals[0])}   # p, box F, box p, dia p
    fn = [lambda a, b: a & b, lambda a, b: a | b, lambda a, b: a & ~b & full, lambda a, b: ~a & b & full]
    for op, arg in uc:
        if op < 16:
            i, d = divmod(op, 4)
            D[d] = vals[i]
        elif op < 80:
            fi, d = divmod(op - 16, 4)
            f, i = divmod(fi, 4)
            D[d] = fn[f](D[d], vals[i])
        elif op < 84:
            D[op - 80] = leaves[arg]
        elif op < 100:
            f, d = divmod(op - 84, 4)
            D[d] = fn[f](D[d], leaves[arg])
        elif op < 116:
            f, d = divmod(op - 100, 4)
            D[d] = fn[f](D[d], D[d + 1])
        elif op < 120:
            D[op - 116] = box(D[op - 116])
        elif op < 124:
            D[op - 120] = dia(D[op - 120])
        elif op == 124:
            return D[0] != full                      # refuted: truth set = D0
        elif op == 125:
            return D[0] != 0                         # refuted: truth set = ~D0
        elif op == 126:
            return (D[0] ^ D[1]) != 0
        elif op == 127:
            return (~(D[0] ^ D[1]) & full) != 0
        elif 128 <= op < 132:
            D[op - 128] = 0
        elif 132 <= op < 136:                        # fused forms (csrc/ucode.h, LOWER_FUSE)
            D[0] = box(vals[op - 132])
        elif 136 <= op < 140:
            D[0] = dia(vals[op - 136])
        elif 140 <= op < 144:
            D[op - 140] = box(leaves[arg])
        elif 144 <= op < 148:
            D[op - 144] = dia(leaves[arg])
        else:
            raise AssertionError(f"bad micro-op {op}")
    raise AssertionError("no FIN op")


def _models(rng, n, k, count):
    out = []
    for _ in range(count):
        f = rng.next_u64() & ((1 << (n * n)) - 1)
        v = rng.next_u64() & ((1 << (k * n)) - 1)
        succ = [(f >> (w * n)) & ((1 << n) - 1) for w in range(n)]
        vals = [(v >> (i * n)) & ((1 << n) - 1) for i in range(k)] + [0] * (4 - k)
        out.append((f, v, succ, vals))
    return out


@pytest.mark.parametrize("mode", [0, 1, 3, 4 | 1, 4 | 3])
def test_lowering_matches_oracle_truth(vol, mode):
    """Refuted-or-not of the lowered program == truth set != W from the oracle, on random models,
    for every leaf mode the kernel instantiations use."""
    rng = W.SplitMix64(2024 + mode)
    sets = [(W.corpus_c1(300), 2), (W.corpus_c2(600)[300:], 2), (W.corpus_c4(300), 3)]
    if not mode & 2:
        sets.append((W.pairs_c5(100)[0], 0))
    for progs, k in sets:
        for c in progs:
            uc, need = kb.debug_lower(c, None, k, mode)
            assert 1 <= need <= 4 and uc[-1][0] in (124, 125)
            if mode & 2:
                assert all(op >= 4 and not (16 <= op < 80 and ((op - 16) // 4) % 4 == 0) for op, _ in uc), \
                    "p_0 must be read through the leaf table in this mode"
            if mode & 4:       # a load never stays in front of a modal operator on the same slot
                for (o1, _), (o2, _) in zip(uc, uc[1:]):
                    assert not (80 <= o1 < 84 and o2 in (116 + o1 - 80, 120 + o1 - 80))
                    assert not (o1 < 16 and o1 % 4 == 0 and o2 in (116, 120))
            for n in (3, 5):
                for f, v, succ, vals in _models(rng, n, k, 5):
                    want = vol.truth(c, n, f, k, v) != [1] * n
                    assert _run_ucode(uc, n, succ, vals) == want, (W.to_text(W.from_postfix(c)), n, f, v)


@pytest.mark.parametrize("mode", [0, 1, 3])
def test_pair_lowering_matches_oracle_truth(vol, mode):
    rng = W.SplitMix64(7 + mode)
    progs, pairs, _ = W.pairs_c5(200)
    extra = W.corpus_c2(60)
    cases = list(zip(extra[:30], extra[30:], [2] * 30))
    if mode != 3:
        cases += [(progs[a], progs[b], 0) for a, b in pairs]
    for a, b, k in cases:
        try:
            uc, need = kb.debug_lower(a, b, k, mode)
        except kb.KripkeError as e:
            assert e.status == kb.EUNSUPPORTED
            continue
        assert uc[-1][0] in (126, 127) and need >= 2
        for n in (4, 6):
            for f, v, succ, vals in _models(rng, n, k, 5):
                want = vol.truth(a, n, f, k, v) != vol.truth(b, n, f, k, v)
                assert _run_ucode(uc, n, succ, vals) == want


def test_lowering_uses_no_slot_for_atom_operands():
    """<= 7-node formulas need at most 2 register-stack slots once atoms are operands; the derived
    leaves make []p, <>p, []F, <>T free."""
    needs = [kb.debug_lower(c, None, 2, 3)[1] for c in W.corpus_c2()]
    assert max(needs) <= 2
    uc, need = kb.debug_lower(W.to_postfix(W.parse("[]p->(<>T&~<>~p)")), None, 2, 3)
    assert need == 1 and all(not (116 <= op < 124) for op, _ in uc)      # no box/dia micro-op left
    uc, need = kb.debug_lower(W.to_postfix(W.parse("[](p->q)->(<>p-><>q)")), None, 2, 3)
    assert need == 2


def test_deep_program_does_not_fit_register_stack():
    deep = W.to_postfix(W.parse("((p&q)|(q&p))&(((p|q)&(q|p))|((p&q)&((q|p)&(p|(q&(p|q))))))"))
    try:
        uc, need = kb.debug_lower(deep, None, 2)
        assert need <= 4
    except kb.KripkeError as e:
        assert e.status == kb.EUNSUPPORTED
    # a perfectly balanced tree of 32 leaves needs 5 slots (atoms are operands): must be refused
    t = [("var", i % 2) for i in range(32)]
    ops = ["and", "or"]
    lvl = 0
    while len(t) > 1:
        t = [(ops[lvl % 2], t[i], t[i + 1]) for i in range(0, len(t), 2)]
        lvl += 1
    with pytest.raises(kb.KripkeError) as e:
        kb.debug_lower(W.to_postfix(t[0]), None, 2)
    assert e.value.status == kb.EUNSUPPORTED


def test_no_cpu_fallback_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    code, offs = W.pack_programs(W.corpus_c1(4))
    with pytest.raises(kb.KripkeError) as e:
        kb.Programs(code, offs, 2)
    assert e.value.status == kb.ECUDA
    with pytest.raises(kb.KripkeError) as e:
        kb.eval_batch_host(code, offs, 3, 2, 0)
    assert e.value.status == kb.ECUDA


def test_bench_starts_one_rank_per_gpu_by_itself():
    """`python bench.py --gpus 2` without a launcher re-executes itself under torch.distributed.run with two
    ranks (one process per GPU).  On a box without a CUDA device both ranks must say so - there is
    no CPU fallback (the launcher's failure report proves the run went through it) - and a rank count that differs from --gpus is refused rather than mislabelled."""
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available():
        pytest.skip("checks the no-device message; on a GPU box the driver's own bench runs cover the launcher")
    bench = os.path.join(ROOT, "bench.py")
    r = subprocess.run([sys.executable, bench, "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and not r.stdout.strip().startswith("{")
    # the launcher stops the other rank as soon as one has failed, so only one of the two messages is certain
    assert re.search(r"no CUDA device on rank [01]", r.stderr + r.stdout)
    assert "torch.distributed" in r.stderr or "torchrun" in r.stderr or "ChildFailedError" in r.stderr
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, bench, "--gpus", "1"], capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode != 0 and "the launcher started 2 rank(s)" in r.stderr
