"""Thin ctypes binding of libkripke_b200.so (include/kripke.h).  Argument marshalling only.

Every function has the name of the C entry point without the `kripke_` prefix.  Device buffers are
torch CUDA tensors (torch is used for device memory and streams only); results come back as the
tensors the C library wrote.  There is no CPU fallback: if the library is missing or no CUDA device
is present the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkripke_b200.so")

OK, EINVAL, EPROGRAM, EUNSUPPORTED, ECUDA, ENOMEM = 0, -1, -2, -3, -4, -5
CLASS_K, CLASS_T, CLASS_S4, CLASS_S5 = 0, 1, 2, 3
ACCUMULATE = 1 << 0
FULL_SWEEP = 1 << 1
NO_SHARING = 1 << 2
NO_SUBTERM_SHARING = 1 << 3
NO_GUARDED_ROOTS = 1 << 10
NO_BOX_DISTRIBUTION = 1 << 11
KERNEL_AUTO, KERNEL_SCALAR, KERNEL_SLICED, KERNEL_JIT = 0 << 4, 1 << 4, 2 << 4, 3 << 4
REDUCE_BLOCK, REDUCE_WARP, REDUCE_THREAD = 0 << 8, 1 << 8, 2 << 8
NO_WITNESS = (1 << 64) - 1

_STATUS = {EINVAL: "KRIPKE_EINVAL", EPROGRAM: "KRIPKE_EPROGRAM", EUNSUPPORTED: "KRIPKE_EUNSUPPORTED",
           ECUDA: "KRIPKE_ECUDA", ENOMEM: "KRIPKE_ENOMEM"}

EXPORTS = [
    "kripke_version", "kripke_last_cuda_error", "kripke_validate_programs", "kripke_programs_create",
    "kripke_programs_destroy", "kripke_class_size", "kripke_eval_batch", "kripke_eval_batch_range",
    "kripke_distinguish_pairs", "kripke_eval_batch_host", "kripke_last_run_info",
    "kripke_calibrate_int32", "kripke_debug_lower", "kripke_witness_to_keys", "kripke_keys_to_witness",
    "kripke_minimal_refutation", "kripke_pairs_separation",
    "kripke_eval_frames", "kripke_distinguish_pairs_frames",
    "kripke_validity_bitmap", "kripke_condition_bitmap", "kripke_match_bitmaps", "kripke_frames_from_bitmap",
    "kripke_failure_density", "kripke_failure_density_frames",
    "kripke_jit_configure", "kripke_debug_jit_source", "kripke_debug_dag_truth", "kripke_signatures", "kripke_frames_generate",
    "kripke_debug_batch_refuted", "kripke_eval_batch_static",
    "kripke_jit_cache_clear",
]


class KripkeError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        extra = f" (cudaError {cuda_error})" if status == ECUDA else ""
        super().__init__(f"{where}: {_STATUS.get(status, status)}{extra}")


class RunInfo(ctypes.Structure):
    _fields_ = [("launches", ctypes.c_uint32), ("kernel_family", ctypes.c_uint32),
                ("sliced_logic_ops_per_word", ctypes.c_uint64), ("models_per_program", ctypes.c_uint64),
                ("executed_models", ctypes.c_uint64), ("logic_instr_per_frame", ctypes.c_double),
                ("jit_programs", ctypes.c_uint32), ("reserved", ctypes.c_uint32),
                ("popc_instr_per_frame", ctypes.c_double),
                ("algorithmic_logic_instr_per_frame", ctypes.c_double),
                ("jit_compile_seconds", ctypes.c_double)]


_lib = None


def load():
    """Loads the library (building it with nvcc first if the .so is not there yet)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from . import build as _build
        _build.build()
    lib = ctypes.CDLL(LIB_PATH)
    vp, u8p, u32p, u64p = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
    u32, u64 = ctypes.c_uint32, ctypes.c_uint64
    lib.kripke_version.restype = ctypes.c_char_p
    lib.kripke_last_cuda_error.restype = ctypes.c_int
    lib.kripke_validate_programs.argtypes = [u8p, u32p, u32, u32, ctypes.POINTER(u32)]
    lib.kripke_programs_create.argtypes = [u8p, u32p, u32, u32, ctypes.POINTER(vp)]
    lib.kripke_programs_destroy.argtypes = [vp]
    lib.kripke_class_size.argtypes = [u32, u32, ctypes.POINTER(u64)]
    lib.kripke_eval_batch.argtypes = [vp, u32, u32, u32, vp, vp, vp]
    lib.kripke_eval_batch_range.argtypes = [vp, u32, u32, u32, u64, u64, u32, vp, vp, vp]
    lib.kripke_distinguish_pairs.argtypes = [vp, u32p, u32, u32, u32, u32, u64, u64, u32, vp, vp, vp]
    lib.kripke_eval_batch_host.argtypes = [u8p, u32p, u32, u32, u32, u32, vp, vp]
    lib.kripke_last_run_info.argtypes = [vp, ctypes.POINTER(RunInfo)]
    lib.kripke_calibrate_int32.argtypes = [u32, ctypes.POINTER(ctypes.c_double),
                                           ctypes.POINTER(ctypes.c_double), vp]
    lib.kripke_minimal_refutation.argtypes = [vp, u32, u32, u32, vp, vp, vp, vp]
    lib.kripke_pairs_separation.argtypes = [vp, u32p, u32, u32, u32, u64, vp, vp, vp]
    lib.kripke_witness_to_keys.argtypes = [vp, u32, u32, u32, vp, vp]
    lib.kripke_keys_to_witness.argtypes = [vp, u32, u32, u32, vp, vp]
    lib.kripke_debug_lower.argtypes = [u8p, u32, u8p, u32, u32, u32, u8p, u32, ctypes.POINTER(u32)]
    lib.kripke_validity_bitmap.argtypes = [vp, u32, u32, u32, u64, u64, vp, vp]
    lib.kripke_condition_bitmap.argtypes = [u32, u32, u32, u64, u64, vp, vp]
    lib.kripke_match_bitmaps.argtypes = [vp, u32, u64, vp, u32, vp, vp]
    lib.kripke_failure_density.argtypes = [vp, u32, u32, u32, u64, u64, vp, vp]
    lib.kripke_failure_density_frames.argtypes = [vp, u32, u32, vp, u64, vp, vp]
    lib.kripke_frames_from_bitmap.argtypes = [u32, u32, u64, u64, vp, vp, u64, vp, vp]
    lib.kripke_eval_frames.argtypes = [vp, u32, u32, vp, u64, u64, u32, vp, vp, vp]
    lib.kripke_distinguish_pairs_frames.argtypes = [vp, u32p, u32, u32, u32, vp, u64, u64, u32, vp, vp, vp]
    lib.kripke_jit_configure.argtypes = [u32, u32]
    lib.kripke_jit_cache_clear.argtypes = [ctypes.POINTER(u32)]
    lib.kripke_signatures.argtypes = [vp, u32, u32, vp, vp]
    lib.kripke_frames_generate.argtypes = [u32, u32, u64, u64, vp, vp]
    lib.kripke_debug_jit_source.argtypes = [u8p, u32p, u32, u32, u32p, u32, u32, u32, u32, u32, u32, ctypes.c_int, vp, u64,
                                            ctypes.POINTER(u32), ctypes.POINTER(u64), ctypes.POINTER(u64)]
    lib.kripke_debug_dag_truth.argtypes = [u8p, u32, u32, u32, u32p, u32p, ctypes.POINTER(u32)]
    lib.kripke_debug_batch_refuted.argtypes = [vp, vp, u32, u32, u32, u32, u32, vp, vp, vp]
    lib.kripke_eval_batch_static.argtypes = [u8p, u32p, u32, u32, u32, u32, u64, u64, u32, vp, vp, vp]
    for name in EXPORTS:
        if name not in ("kripke_version",):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def _check(rc: int, where: str):
    if rc != OK:
        raise KripkeError(rc, where, load().kripke_last_cuda_error())


def _host(code, offsets):
    code = np.ascontiguousarray(code, dtype=np.uint8)
    offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
    if code.size == 0:
        code = np.zeros(1, np.uint8)
    return code, offsets


def version() -> str:
    return load().kripke_version().decode()


def validate_programs(code, offsets, n_vars: int) -> int:
    """Returns the deepest postfix stack any program needs; raises KripkeError if invalid."""
    code, offsets = _host(code, offsets)
    deepest = ctypes.c_uint32(0)
    _check(load().kripke_validate_programs(code.ctypes.data, offsets.ctypes.data, len(offsets) - 1,
                                           n_vars, ctypes.byref(deepest)), "kripke_validate_programs")
    return deepest.value


def class_size(n_worlds: int, frame_class: int) -> int:
    out = ctypes.c_uint64(0)
    _check(load().kripke_class_size(n_worlds, frame_class, ctypes.byref(out)), "kripke_class_size")
    return out.value


class Programs:
    """Owner of a kripke_programs_t handle."""

    def __init__(self, code, offsets, n_vars: int):
        code, offsets = _host(code, offsets)
        self.n_formulas = len(offsets) - 1
        self.n_vars = n_vars
        self._h = ctypes.c_void_p()
        _check(load().kripke_programs_create(code.ctypes.data, offsets.ctypes.data, self.n_formulas,
                                             n_vars, ctypes.byref(self._h)), "kripke_programs_create")

    def destroy(self):
        if self._h:
            load().kripke_programs_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def last_run_info(self) -> RunInfo:
        info = RunInfo()
        _check(load().kripke_last_run_info(self._h, ctypes.byref(info)), "kripke_last_run_info")
        return info


def programs_create(code, offsets, n_vars: int) -> Programs:
    return Programs(code, offsets, n_vars)


def programs_destroy(p: Programs):
    p.destroy()


def _outputs(n: int, counts_out, witness_out):
    import torch
    if counts_out is None:
        counts_out = torch.empty((n, 2), dtype=torch.int64, device="cuda")
    if witness_out is None:
        witness_out = torch.empty((n, 2), dtype=torch.int64, device="cuda")
    for t in (counts_out, witness_out):
        assert t.is_cuda and t.dtype == torch.int64 and t.is_contiguous() and t.numel() >= 2 * n
    return counts_out, witness_out


def _stream(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def eval_batch(programs: Programs, n_worlds: int, n_vars: int, frame_class: int,
               counts_out=None, witness_out=None, stream=None):
    """kripke_eval_batch.  Returns (counts, witness): int64 CUDA tensors of shape (B, 2) holding the
    kripke_count_t / kripke_witness_t records (see unpack())."""
    counts_out, witness_out = _outputs(programs.n_formulas, counts_out, witness_out)
    _check(load().kripke_eval_batch(programs._h, n_worlds, n_vars, frame_class, counts_out.data_ptr(),
                                    witness_out.data_ptr(), _stream(stream)), "kripke_eval_batch")
    return counts_out, witness_out


def eval_batch_range(programs: Programs, n_worlds: int, n_vars: int, frame_class: int,
                     frame_begin: int, frame_count: int, flags: int = 0,
                     counts_out=None, witness_out=None, stream=None):
    counts_out, witness_out = _outputs(programs.n_formulas, counts_out, witness_out)
    _check(load().kripke_eval_batch_range(programs._h, n_worlds, n_vars, frame_class, frame_begin,
                                          frame_count, flags, counts_out.data_ptr(),
                                          witness_out.data_ptr(), _stream(stream)),
           "kripke_eval_batch_range")
    return counts_out, witness_out


def jit_cache_clear() -> int:
    """kripke_jit_cache_clear: forget every cached plan and unload every compiled module (no Programs object
    may be alive).  Returns the number of modules unloaded."""
    n = ctypes.c_uint32(0)
    _check(load().kripke_jit_cache_clear(ctypes.byref(n)), "kripke_jit_cache_clear")
    return n.value


STATIC_MAX_FORMULAS = 8192
STATIC_MAX_CLASS_FRAMES = 8192
STATIC_SCRATCH_BYTES = 819456


def eval_batch_static(code, offsets, n_worlds: int, n_vars: int, frame_class: int, frame_begin: int,
                      frame_count: int, counts_out, witness_out, flags: int = 0, stream=None):
    """kripke_eval_batch_static: the scan for callers that cannot allocate device memory (their memory
    belongs to another pool, or they cannot take cudaMalloc's device-wide synchronisation).  No handle:
    code / offsets are the HOST program arrays, counts_out / witness_out the caller's own int64 CUDA
    tensors of shape (B, 2) - unlike the other wrappers this one never creates a tensor, so the call
    allocates nothing on the device.  Working memory is the library's fixed static block; calls that
    overlap on the GPU race on it."""
    code, offsets = _host(code, offsets)
    n = len(offsets) - 1
    assert counts_out is not None and witness_out is not None, "the caller provides the output tensors"
    _outputs(n, counts_out, witness_out)
    _check(load().kripke_eval_batch_static(code.ctypes.data, offsets.ctypes.data, n, n_worlds, n_vars,
                                           frame_class, frame_begin, frame_count, flags,
                                           counts_out.data_ptr(), witness_out.data_ptr(), _stream(stream)),
           "kripke_eval_batch_static")
    return counts_out, witness_out


def distinguish_pairs(programs: Programs, pairs, n_worlds: int, n_vars: int, frame_class: int,
                      frame_begin: int, frame_count: int, flags: int = 0,
                      counts_out=None, witness_out=None, stream=None):
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1)
    n_pairs = len(pairs) // 2
    counts_out, witness_out = _outputs(n_pairs, counts_out, witness_out)
    _check(load().kripke_distinguish_pairs(programs._h, pairs.ctypes.data, n_pairs, n_worlds, n_vars,
                                           frame_class, frame_begin, frame_count, flags,
                                           counts_out.data_ptr(), witness_out.data_ptr(),
                                           _stream(stream)), "kripke_distinguish_pairs")
    return counts_out, witness_out


def _succ(succ, n_worlds: int):
    """succ: CUDA tensor of successor masks, int16 (bit pattern of uint16) or uint16, F*n entries."""
    import torch
    assert succ.is_cuda and succ.is_contiguous() and succ.element_size() == 2
    assert succ.numel() % n_worlds == 0
    return succ.numel() // n_worlds


def eval_frames(programs: Programs, n_worlds: int, n_vars: int, succ, index_base: int = 0, flags: int = 0,
                counts_out=None, witness_out=None, stream=None):
    """kripke_eval_frames: every program on every listed frame (succ: CUDA tensor of F*n 16-bit
    successor masks) and every valuation.  witness.frame = index_base + list position."""
    n_frames = _succ(succ, n_worlds)
    counts_out, witness_out = _outputs(programs.n_formulas, counts_out, witness_out)
    _check(load().kripke_eval_frames(programs._h, n_worlds, n_vars, succ.data_ptr(), n_frames, index_base,
                                     flags, counts_out.data_ptr(), witness_out.data_ptr(), _stream(stream)),
           "kripke_eval_frames")
    return counts_out, witness_out


def distinguish_pairs_frames(programs: Programs, pairs, n_worlds: int, n_vars: int, succ,
                             index_base: int = 0, flags: int = 0, counts_out=None, witness_out=None,
                             stream=None):
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1)
    n_pairs = len(pairs) // 2
    n_frames = _succ(succ, n_worlds)
    counts_out, witness_out = _outputs(n_pairs, counts_out, witness_out)
    _check(load().kripke_distinguish_pairs_frames(programs._h, pairs.ctypes.data, n_pairs, n_worlds, n_vars,
                                                  succ.data_ptr(), n_frames, index_base, flags,
                                                  counts_out.data_ptr(), witness_out.data_ptr(),
                                                  _stream(stream)), "kripke_distinguish_pairs_frames")
    return counts_out, witness_out


COND = {"reflexive": 0, "transitive": 1, "symmetric": 2, "serial": 3, "euclidean": 4,
        "partially_functional": 5, "dense": 6, "confluent": 7}


def validity_bitmap(programs: Programs, n_worlds: int, n_vars: int, frame_class: int, frame_begin: int,
                    frame_count: int, bitmap_out=None, stream=None):
    """kripke_validity_bitmap.  Returns an int32 CUDA tensor (B, ceil(frame_count/32)) of bit words."""
    import torch
    words = (frame_count + 31) // 32
    if bitmap_out is None:
        bitmap_out = torch.zeros((programs.n_formulas, words), dtype=torch.int32, device="cuda")
    assert bitmap_out.is_cuda and bitmap_out.is_contiguous() and bitmap_out.numel() >= programs.n_formulas * words
    _check(load().kripke_validity_bitmap(programs._h, n_worlds, n_vars, frame_class, frame_begin, frame_count,
                                         bitmap_out.data_ptr(), _stream(stream)), "kripke_validity_bitmap")
    return bitmap_out


def condition_bitmap(n_worlds: int, condition: int, frame_class: int, frame_begin: int, frame_count: int,
                     bitmap_out=None, stream=None):
    import torch
    words = (frame_count + 31) // 32
    if bitmap_out is None:
        bitmap_out = torch.zeros((words,), dtype=torch.int32, device="cuda")
    assert bitmap_out.is_cuda and bitmap_out.is_contiguous() and bitmap_out.numel() >= words
    _check(load().kripke_condition_bitmap(n_worlds, condition, frame_class, frame_begin, frame_count,
                                          bitmap_out.data_ptr(), _stream(stream)), "kripke_condition_bitmap")
    return bitmap_out


def match_bitmaps(bitmaps, library, match_out=None, stream=None):
    """kripke_match_bitmaps: bitmaps (R, words), library (L, words) int32 CUDA tensors -> int32 (R,)
    index of the first equal library row, -1 if none."""
    import torch
    assert bitmaps.is_cuda and library.is_cuda and bitmaps.is_contiguous() and library.is_contiguous()
    n_records, words = bitmaps.shape
    assert library.shape[1] == words
    if match_out is None:
        match_out = torch.empty((n_records,), dtype=torch.int32, device="cuda")
    _check(load().kripke_match_bitmaps(bitmaps.data_ptr(), n_records, words, library.data_ptr(), library.shape[0],
                                       match_out.data_ptr(), _stream(stream)), "kripke_match_bitmaps")
    return match_out


def frames_from_bitmap(n_worlds: int, frame_class: int, frame_begin: int, frame_count: int, bitmap, capacity: int,
                       stream=None):
    """kripke_frames_from_bitmap.  Returns (succ int16 CUDA tensor of capacity*n masks, number of set bits);
    synchronises to read the count."""
    import torch
    succ = torch.zeros((max(1, capacity) * n_worlds,), dtype=torch.int16, device="cuda")
    count = torch.zeros((1,), dtype=torch.int64, device="cuda")
    _check(load().kripke_frames_from_bitmap(n_worlds, frame_class, frame_begin, frame_count, bitmap.data_ptr(),
                                            succ.data_ptr(), capacity, count.data_ptr(), _stream(stream)),
           "kripke_frames_from_bitmap")
    n_set = int(count.item())
    return succ[:min(n_set, capacity) * n_worlds], n_set


def failure_density(programs: Programs, n_worlds: int, n_vars: int, frame_class: int, frame_begin: int,
                    frame_count: int, counts_out=None, stream=None):
    """kripke_failure_density.  Returns an int32 CUDA tensor (B, frame_count) of failing (valuation, world)
    pair counts."""
    import torch
    if counts_out is None:
        counts_out = torch.zeros((programs.n_formulas, frame_count), dtype=torch.int32, device="cuda")
    assert counts_out.is_cuda and counts_out.is_contiguous() and counts_out.numel() >= programs.n_formulas * frame_count
    _check(load().kripke_failure_density(programs._h, n_worlds, n_vars, frame_class, frame_begin, frame_count,
                                         counts_out.data_ptr(), _stream(stream)), "kripke_failure_density")
    return counts_out


def failure_density_frames(programs: Programs, n_worlds: int, n_vars: int, succ, counts_out=None, stream=None):
    import torch
    n_frames = _succ(succ, n_worlds)
    if counts_out is None:
        counts_out = torch.zeros((programs.n_formulas, n_frames), dtype=torch.int32, device="cuda")
    assert counts_out.is_cuda and counts_out.is_contiguous() and counts_out.numel() >= programs.n_formulas * n_frames
    _check(load().kripke_failure_density_frames(programs._h, n_worlds, n_vars, succ.data_ptr(), n_frames,
                                                counts_out.data_ptr(), _stream(stream)),
           "kripke_failure_density_frames")
    return counts_out


GEN_TEMPLATES, GEN_ERDOS_RENYI, GEN_EDGE_FLIP, GEN_DEAD_END, GEN_BACK_EDGE, GEN_STRESS = range(6)


def frames_generate(generator: int, n_worlds: int, n_frames: int, seed: int, succ_out=None, stream=None):
    """kripke_frames_generate: int16 CUDA tensor of n_frames * n_worlds successor masks (bit pattern of uint16)."""
    import torch
    if succ_out is None:
        succ_out = torch.empty((max(1, n_frames) * n_worlds,), dtype=torch.int16, device="cuda")[:n_frames * n_worlds]
    _check(load().kripke_frames_generate(generator, n_worlds, n_frames, seed, succ_out.data_ptr(), _stream(stream)),
           "kripke_frames_generate")
    return succ_out


def signatures(programs: Programs, n_vars: int, n_max: int = 3, sig_out=None, stream=None):
    """kripke_signatures: int64 CUDA tensor (B, 2) holding the two 64-bit sums per formula."""
    import torch
    if sig_out is None:
        sig_out = torch.empty((programs.n_formulas, 2), dtype=torch.int64, device="cuda")
    _check(load().kripke_signatures(programs._h, n_vars, n_max, sig_out.data_ptr(), _stream(stream)), "kripke_signatures")
    return sig_out


def bits_to_bool(bitmap, count: int):
    """int32 bit words (..., words) (torch or numpy) -> numpy bool array (..., count)."""
    a = bitmap.cpu().numpy() if hasattr(bitmap, "cpu") else np.asarray(bitmap)
    a = np.ascontiguousarray(a).view(np.uint32)
    bits = (a[..., :, None] >> np.arange(32, dtype=np.uint32)) & 1
    return bits.reshape(a.shape[:-1] + (-1,))[..., :count].astype(bool)


def minimal_refutation(programs: Programs, n_vars: int, frame_class: int, n_max: int,
                       size_out=None, counts_out=None, witness_out=None, stream=None):
    """kripke_minimal_refutation.  Returns (size int32 (B,), counts int64 (B,2), witness int64 (B,2))
    CUDA tensors; size 0 = no countermodel through n_max worlds."""
    import torch
    n = programs.n_formulas
    if size_out is None:
        size_out = torch.empty((n,), dtype=torch.int32, device="cuda")
    counts_out, witness_out = _outputs(n, counts_out, witness_out)
    _check(load().kripke_minimal_refutation(programs._h, n_vars, frame_class, n_max, size_out.data_ptr(),
                                            counts_out.data_ptr(), witness_out.data_ptr(), _stream(stream)),
           "kripke_minimal_refutation")
    return size_out, counts_out, witness_out


def pairs_separation(programs: Programs, pairs, n_vars: int, n_max: int, chunk_frames: int = 1 << 30,
                     stream=None):
    """kripke_pairs_separation.  Returns (size uint32 (P,), witness uint64 (P,2)) numpy arrays."""
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1)
    n_pairs = len(pairs) // 2
    size = np.zeros(n_pairs, np.uint32)
    witness = np.zeros((n_pairs, 2), np.uint64)
    _check(load().kripke_pairs_separation(programs._h, pairs.ctypes.data, n_pairs, n_vars, n_max,
                                          chunk_frames, size.ctypes.data, witness.ctypes.data,
                                          _stream(stream)), "kripke_pairs_separation")
    return size, witness


def eval_batch_host(code, offsets, n_worlds: int, n_vars: int, frame_class: int):
    """kripke_eval_batch_host: host buffers in, host buffers out (numpy uint64 arrays (B, 2))."""
    code, offsets = _host(code, offsets)
    n = len(offsets) - 1
    counts = np.zeros((n, 2), np.uint64)
    witness = np.zeros((n, 2), np.uint64)
    _check(load().kripke_eval_batch_host(code.ctypes.data, offsets.ctypes.data, n, n_worlds, n_vars,
                                         frame_class, counts.ctypes.data, witness.ctypes.data),
           "kripke_eval_batch_host")
    return counts, witness


def calibrate_int32(variant: int = 0, stream=None):
    """Returns (thread-instructions per second, elapsed ms) of the integer-pipe calibration."""
    rate, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(load().kripke_calibrate_int32(variant, ctypes.byref(rate), ctypes.byref(ms), _stream(stream)),
           "kripke_calibrate_int32")
    return rate.value, ms.value


def witness_to_keys(witness, n_worlds: int, n_vars: int, keys_out=None, stream=None):
    """Device witness records (int64 (B, 2) CUDA tensor) -> int64 (B,) keys whose MIN is the
    lexicographically first (frame, valuation)."""
    import torch
    n = witness.shape[0]
    if keys_out is None:
        keys_out = torch.empty((n,), dtype=torch.int64, device="cuda")
    _check(load().kripke_witness_to_keys(witness.data_ptr(), n, n_worlds, n_vars, keys_out.data_ptr(),
                                         _stream(stream)), "kripke_witness_to_keys")
    return keys_out


def keys_to_witness(keys, n_worlds: int, n_vars: int, witness_out=None, stream=None):
    import torch
    n = keys.shape[0]
    if witness_out is None:
        witness_out = torch.empty((n, 2), dtype=torch.int64, device="cuda")
    _check(load().kripke_keys_to_witness(keys.data_ptr(), n, n_worlds, n_vars, witness_out.data_ptr(),
                                         _stream(stream)), "kripke_keys_to_witness")
    return witness_out


def debug_lower(code_a: bytes, code_b: bytes | None, n_vars: int, leaf_mode: int = 0):
    """([(op, arg), ...], register-stack slots needed); raises KripkeError(EUNSUPPORTED) if the
    program does not fit the bit-sliced kernel."""
    a = np.frombuffer(bytes(code_a), np.uint8).copy()
    b = np.frombuffer(bytes(code_b), np.uint8).copy() if code_b is not None else None
    out = np.zeros(256, np.uint16)
    need = ctypes.c_uint32(0)
    rc = load().kripke_debug_lower(a.ctypes.data, len(a), b.ctypes.data if b is not None else None,
                                   len(b) if b is not None else 0, n_vars, leaf_mode, out.ctypes.data,
                                   len(out), ctypes.byref(need))
    if rc < 0:
        raise KripkeError(rc, "kripke_debug_lower")
    return [(int(x) & 0xFF, int(x) >> 8) for x in out[:rc]], need.value



def jit_configure(max_programs_per_kernel: int = 64, min_blocks_per_sm: int = 2):
    _check(load().kripke_jit_configure(max_programs_per_kernel, min_blocks_per_sm), "kripke_jit_configure")


def debug_jit_source(code, offsets, n_vars: int, n_worlds: int, frame_class: int, group_vars: int,
                     kernel_index: int = 0, flags: int = 0, pairs=None, compile: bool = False, density: bool = False):
    """(source text, kernels in the group, logic ops per word of this kernel, cubin bytes) of one compiled
    kernel; None if the emitter has no layout for the shape.  Pure host."""
    code, offsets = _host(code, offsets)
    cap = 1 << 22
    buf = ctypes.create_string_buffer(cap)
    nk, ops, cb = ctypes.c_uint32(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
    pa = None if pairs is None else np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1)
    rc = load().kripke_debug_jit_source(code.ctypes.data, offsets.ctypes.data, len(offsets) - 1, n_vars,
                                        None if pa is None else pa.ctypes.data,
                                        0 if pa is None else len(pa) // 2, n_worlds, frame_class, flags, group_vars,
                                        kernel_index, (1 if compile else 0) | (2 if density else 0),
                                        ctypes.cast(buf, ctypes.c_void_p), cap,
                                        ctypes.byref(nk), ctypes.byref(ops), ctypes.byref(cb))
    if rc == EUNSUPPORTED:
        return None
    if rc < 0:
        raise KripkeError(rc, "kripke_debug_jit_source")
    return buf.value.decode(), nk.value, ops.value, cb.value


def debug_batch_refuted(code, offsets, n_vars: int, n_worlds: int, frame_class: int, succ, val, flags: int = 0):
    """(refuted flag per formula, rewrites applied): does the model refute each formula, evaluated on the forms
    the compiled kernels evaluate (guarded roots, redistributed boxes, canonical variable order)?  Pure host."""
    code, offsets = _host(code, offsets)
    s = np.ascontiguousarray(succ, dtype=np.uint32)
    v = np.ascontiguousarray(list(val) + [0] * (4 - len(val)), dtype=np.uint32)
    out = np.zeros(len(offsets) - 1, dtype=np.uint8)
    rc = load().kripke_debug_batch_refuted(code.ctypes.data, offsets.ctypes.data, len(offsets) - 1, n_vars, n_worlds,
                                           frame_class, flags, s.ctypes.data, v.ctypes.data, out.ctypes.data)
    if rc < 0:
        raise KripkeError(rc, "kripke_debug_batch_refuted")
    return out.astype(bool), rc


def debug_dag_truth(code: bytes, n_vars: int, n_worlds: int, succ, val) -> int:
    """Truth set (bit mask) of one program on one model as the compiled scans' batch graph computes it."""
    a = np.frombuffer(code, dtype=np.uint8)
    s = np.ascontiguousarray(succ, dtype=np.uint32)
    v = np.ascontiguousarray(list(val) + [0] * (4 - len(val)), dtype=np.uint32)
    out = ctypes.c_uint32(0)
    rc = load().kripke_debug_dag_truth(a.ctypes.data, len(a), n_vars, n_worlds, s.ctypes.data, v.ctypes.data,
                                       ctypes.byref(out))
    if rc < 0:
        raise KripkeError(rc, "kripke_debug_dag_truth")
    return out.value


def unpack(counts, witness):
    """(counts, witness) as returned above (torch or numpy) -> dict of numpy uint64/uint32 arrays:
    models, frames, wit_f (NO_WITNESS = none), wit_v, wit_w."""
    if hasattr(counts, "cpu"):
        counts = counts.cpu().numpy()
        witness = witness.cpu().numpy()
    c = np.ascontiguousarray(counts).view(np.uint64).reshape(-1, 2)
    w = np.ascontiguousarray(witness).view(np.uint64).reshape(-1, 2)
    return {"models": c[:, 0].copy(), "frames": c[:, 1].copy(), "wit_f": w[:, 0].copy(),
            "wit_v": (w[:, 1] & np.uint64(0xFFFFFFFF)).astype(np.uint32),
            "wit_w": (w[:, 1] >> np.uint64(32)).astype(np.uint32)}
