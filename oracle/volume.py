"""ctypes front end of oracle/volume_oracle.c.  TEST INFRASTRUCTURE (see that file's header).

`build()` compiles the C file with gcc into oracle/libkripke_oracle.so (git-ignored); every entry
point below loads it lazily.  Nothing here touches the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "volume_oracle.c")
_LIB = os.path.join(_HERE, "libkripke_oracle.so")
_lib = None

NO_WITNESS = (1 << 64) - 1
CLASS_K, CLASS_T, CLASS_S4, CLASS_S5 = 0, 1, 2, 3
COND = {"reflexive": 0, "transitive": 1, "symmetric": 2, "serial": 3, "euclidean": 4,
        "partially_functional": 5, "dense": 6, "confluent": 7}


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O3", "-march=native", "-std=c99", "-fopenmp", "-shared", "-fPIC",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u8p = ctypes.POINTER(ctypes.c_uint8)
        u32p = ctypes.POINTER(ctypes.c_uint32)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        lib.kov_count_condition.restype = ctypes.c_uint64
        lib.kov_count_condition.argtypes = [ctypes.c_int, ctypes.c_int]
        lib.kov_condition_bitmap.restype = ctypes.c_int
        lib.kov_condition_bitmap.argtypes = [ctypes.c_int, ctypes.c_int, u8p]
        lib.kov_class_frames.restype = ctypes.c_int64
        lib.kov_class_frames.argtypes = [ctypes.c_int, ctypes.c_int, u64p, ctypes.c_uint64]
        lib.kov_truth.restype = ctypes.c_int
        lib.kov_truth.argtypes = [u8p, ctypes.c_uint32, ctypes.c_int, ctypes.c_uint64, ctypes.c_int,
                                  ctypes.c_uint64, u8p]
        lib.kov_census_list.restype = ctypes.c_int
        lib.kov_census_list.argtypes = [u8p, u32p, ctypes.c_uint32, u32p, ctypes.c_uint32,
                                        ctypes.c_int, ctypes.c_int, u64p, u64p, ctypes.c_uint64,
                                        u64p, u64p, u64p, u32p, u32p, ctypes.c_int]
        lib.kov_census_relations.restype = ctypes.c_int
        lib.kov_census_relations.argtypes = [u8p, u32p, ctypes.c_uint32, u32p, ctypes.c_uint32,
                                             ctypes.c_int, ctypes.c_int, u8p, ctypes.c_uint64,
                                             u64p, u64p, u64p, u32p, u32p, ctypes.c_int]
        lib.kov_validity_list.restype = ctypes.c_int
        lib.kov_validity_list.argtypes = [u8p, u32p, ctypes.c_uint32, ctypes.c_int, ctypes.c_int, u64p,
                                          ctypes.c_uint64, u8p, ctypes.c_int]
        lib.kov_failure_counts.restype = ctypes.c_int
        lib.kov_failure_counts.argtypes = [u8p, u32p, ctypes.c_uint32, ctypes.c_int, ctypes.c_int, u64p,
                                           ctypes.c_uint64, u32p, ctypes.c_int]
        lib.kov_failure_counts_relations.restype = ctypes.c_int
        lib.kov_failure_counts_relations.argtypes = [u8p, u32p, ctypes.c_uint32, ctypes.c_int, ctypes.c_int, u8p,
                                                     ctypes.c_uint64, u32p, ctypes.c_int]
        lib.kov_max_threads.restype = ctypes.c_int
        lib.kov_orbits.restype = ctypes.c_int64
        lib.kov_orbits.argtypes = [ctypes.c_int, u64p, u64p, ctypes.c_uint64]
        lib.kov_signatures.restype = ctypes.c_int
        lib.kov_signatures.argtypes = [u8p, u32p, ctypes.c_uint32, ctypes.c_int, ctypes.c_int, u64p, u64p]
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def max_threads() -> int:
    return int(_load().kov_max_threads())


def count_condition(n: int, cond: str) -> int:
    return int(_load().kov_count_condition(n, COND[cond]))


def condition_bitmap(n: int, cond: str) -> np.ndarray:
    out = np.zeros(1 << (n * n), dtype=np.uint8)
    rc = _load().kov_condition_bitmap(n, COND[cond], _p(out, ctypes.c_uint8))
    if rc:
        raise ValueError("kov_condition_bitmap failed")
    return out


_class_cache = {}


def class_frames(n: int, cls: int) -> np.ndarray:
    """Ascending K-indices of the class members (uint64)."""
    key = (n, cls)
    if key not in _class_cache:
        lib = _load()
        cnt = lib.kov_class_frames(n, cls, None, 0)
        if cnt < 0:
            raise ValueError("kov_class_frames failed")
        out = np.zeros(cnt, dtype=np.uint64)
        lib.kov_class_frames(n, cls, _p(out, ctypes.c_uint64), cnt)
        _class_cache[key] = out
    return _class_cache[key]


def truth(code: bytes, n: int, f: int, k: int, v: int) -> list:
    buf = np.frombuffer(bytes(code), dtype=np.uint8).copy()
    out = np.zeros(8, dtype=np.uint8)
    rc = _load().kov_truth(_p(buf, ctypes.c_uint8), len(buf), n, f, k, v, _p(out, ctypes.c_uint8))
    if rc:
        raise ValueError("malformed program")
    return [int(x) for x in out[:n]]


def census_list(code, offsets, n, k, frames, weights=None, pairs=None, threads=0):
    """Census of every program (or every pair) over an explicit list of K-indices.

    Returns a dict of numpy arrays: models, frames (uint64), wit_f (uint64; NO_WITNESS = none),
    wit_v, wit_w (uint32), one entry per formula (or per pair)."""
    code = np.ascontiguousarray(code, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
    frames = np.ascontiguousarray(frames, dtype=np.uint64)
    B = len(offsets) - 1
    if weights is not None:
        weights = np.ascontiguousarray(weights, dtype=np.uint64)
        assert len(weights) == len(frames)
    P = 0
    if pairs is not None:
        pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1)
        P = len(pairs) // 2
        assert pairs.max(initial=0) < B
    Q = P if pairs is not None else B
    res = {"models": np.zeros(Q, np.uint64), "frames": np.zeros(Q, np.uint64),
           "wit_f": np.zeros(Q, np.uint64), "wit_v": np.zeros(Q, np.uint32),
           "wit_w": np.zeros(Q, np.uint32)}
    if len(code) == 0:
        code = np.zeros(1, np.uint8)
    rc = _load().kov_census_list(
        _p(code, ctypes.c_uint8), _p(offsets, ctypes.c_uint32), B,
        _p(pairs, ctypes.c_uint32), P, n, k,
        _p(frames if len(frames) else np.zeros(1, np.uint64), ctypes.c_uint64),
        _p(weights, ctypes.c_uint64), len(frames),
        _p(res["models"], ctypes.c_uint64), _p(res["frames"], ctypes.c_uint64),
        _p(res["wit_f"], ctypes.c_uint64), _p(res["wit_v"], ctypes.c_uint32),
        _p(res["wit_w"], ctypes.c_uint32), threads)
    if rc:
        raise ValueError("kov_census_list failed (malformed program or bad argument)")
    return res


def census_relations(code, offsets, n, k, rel, pairs=None, threads=0):
    """Census of every program (or pair) over explicit frames rel[F, n, n] (uint8 adjacency matrices,
    n <= 16) and all 2^(k*n) valuations.  Same dict as census_list; wit_f is the POSITION in rel."""
    code = np.ascontiguousarray(code, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
    rel = np.ascontiguousarray(rel, dtype=np.uint8)
    assert rel.ndim == 3 and rel.shape[1] == n and rel.shape[2] == n
    B = len(offsets) - 1
    P = 0
    if pairs is not None:
        pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1)
        P = len(pairs) // 2
        assert pairs.max(initial=0) < B
    Q = P if pairs is not None else B
    res = {"models": np.zeros(Q, np.uint64), "frames": np.zeros(Q, np.uint64),
           "wit_f": np.zeros(Q, np.uint64), "wit_v": np.zeros(Q, np.uint32),
           "wit_w": np.zeros(Q, np.uint32)}
    if len(code) == 0:
        code = np.zeros(1, np.uint8)
    rc = _load().kov_census_relations(
        _p(code, ctypes.c_uint8), _p(offsets, ctypes.c_uint32), B, _p(pairs, ctypes.c_uint32), P, n, k,
        _p(rel if len(rel) else np.zeros((1, n, n), np.uint8), ctypes.c_uint8), len(rel),
        _p(res["models"], ctypes.c_uint64), _p(res["frames"], ctypes.c_uint64),
        _p(res["wit_f"], ctypes.c_uint64), _p(res["wit_v"], ctypes.c_uint32),
        _p(res["wit_w"], ctypes.c_uint32), threads)
    if rc:
        raise ValueError("kov_census_relations failed (malformed program or bad argument)")
    return res


def census(code, offsets, n, k, cls=CLASS_K, frame_begin=0, frame_count=None, pairs=None, threads=0):
    """Census over class frames [frame_begin, frame_begin + frame_count) in class order."""
    if cls == CLASS_K:
        total = 1 << (n * n)
        if frame_count is None:
            frame_count = total - frame_begin
        assert frame_begin + frame_count <= total
        frames = np.arange(frame_begin, frame_begin + frame_count, dtype=np.uint64)
    else:
        allf = class_frames(n, cls)
        if frame_count is None:
            frame_count = len(allf) - frame_begin
        frames = allf[frame_begin:frame_begin + frame_count]
    return census_list(code, offsets, n, k, frames, None, pairs, threads)


def validity(code, offsets, n, k, cls=CLASS_K, frame_begin=0, frame_count=None, threads=0):
    """uint8 array [B, frame_count]: 1 iff formula b is valid on the class frame frame_begin + i
    (class order = ascending f): no valuation and no world falsify it."""
    code = np.ascontiguousarray(code, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
    if cls == CLASS_K:
        total = 1 << (n * n)
        if frame_count is None:
            frame_count = total - frame_begin
        frames = np.arange(frame_begin, frame_begin + frame_count, dtype=np.uint64)
    else:
        allf = class_frames(n, cls)
        if frame_count is None:
            frame_count = len(allf) - frame_begin
        frames = np.ascontiguousarray(allf[frame_begin:frame_begin + frame_count], dtype=np.uint64)
    B = len(offsets) - 1
    out = np.zeros((B, len(frames)), np.uint8)
    if len(frames) == 0 or B == 0:
        return out
    rc = _load().kov_validity_list(_p(code, ctypes.c_uint8), _p(offsets, ctypes.c_uint32), B, n, k,
                                   _p(frames, ctypes.c_uint64), len(frames), _p(out, ctypes.c_uint8), threads)
    if rc:
        raise ValueError("kov_validity_list failed")
    return out


def failure_counts(code, offsets, n, k, cls=CLASS_K, frame_begin=0, frame_count=None, rel=None, threads=0):
    """uint32 array [B, frames]: the number of (valuation, world) pairs at which formula b fails on each
    frame (density = count / (2^(k*n) * n)).  Frames: the class range, or - if `rel` is
    given - the explicit relations rel[F, n, n] (n <= 16)."""
    code = np.ascontiguousarray(code, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
    B = len(offsets) - 1
    if rel is not None:
        rel = np.ascontiguousarray(rel, dtype=np.uint8)
        out = np.zeros((B, len(rel)), np.uint32)
        if len(rel) and B:
            rc = _load().kov_failure_counts_relations(_p(code, ctypes.c_uint8), _p(offsets, ctypes.c_uint32), B, n, k,
                                                      _p(rel, ctypes.c_uint8), len(rel), _p(out, ctypes.c_uint32), threads)
            if rc:
                raise ValueError("kov_failure_counts_relations failed")
        return out
    if cls == CLASS_K:
        total = 1 << (n * n)
        if frame_count is None:
            frame_count = total - frame_begin
        frames = np.arange(frame_begin, frame_begin + frame_count, dtype=np.uint64)
    else:
        allf = class_frames(n, cls)
        if frame_count is None:
            frame_count = len(allf) - frame_begin
        frames = np.ascontiguousarray(allf[frame_begin:frame_begin + frame_count], dtype=np.uint64)
    out = np.zeros((B, len(frames)), np.uint32)
    if len(frames) and B:
        rc = _load().kov_failure_counts(_p(code, ctypes.c_uint8), _p(offsets, ctypes.c_uint32), B, n, k,
                                        _p(frames, ctypes.c_uint64), len(frames), _p(out, ctypes.c_uint32), threads)
        if rc:
            raise ValueError("kov_failure_counts failed")
    return out


def signatures(code, offsets, max_n: int, k: int):
    """Per formula, a 128-bit hash (two uint64 arrays) of its truth sets on every model of
    1..max_n worlds; equal signatures <=> equal truth sets on all those models."""
    code = np.ascontiguousarray(code, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
    B = len(offsets) - 1
    a = np.zeros(B, np.uint64)
    b = np.zeros(B, np.uint64)
    rc = _load().kov_signatures(_p(code, ctypes.c_uint8), _p(offsets, ctypes.c_uint32), B, max_n, k,
                                _p(a, ctypes.c_uint64), _p(b, ctypes.c_uint64))
    if rc:
        raise ValueError("kov_signatures failed")
    return a, b


def orbits(n: int):
    """(representatives, sizes): the least K-index of every isomorphism class of n-world frames,
    ascending, and the class sizes (uint64 arrays).  sum(sizes) = 2^(n*n)."""
    lib = _load()
    cnt = lib.kov_orbits(n, None, None, 0)
    if cnt < 0:
        raise ValueError("kov_orbits failed")
    reps = np.zeros(cnt, np.uint64)
    sizes = np.zeros(cnt, np.uint64)
    lib.kov_orbits(n, _p(reps, ctypes.c_uint64), _p(sizes, ctypes.c_uint64), cnt)
    return reps, sizes
