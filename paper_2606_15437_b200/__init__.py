"""B200-native fused bitmask Kripke evaluation (hot path of arxiv/paper_2606_15437).

The product is the C-ABI library `libkripke_b200.so` (include/kripke.h; CUDA sources in csrc/);
`binding` is its thin ctypes front end with the same names.  See DESIGN.md.
"""
from . import binding  # noqa: F401
from .binding import (  # noqa: F401
    KripkeError, Programs, programs_create, programs_destroy, validate_programs, class_size,
    eval_batch, eval_batch_range, distinguish_pairs, eval_batch_host, calibrate_int32, unpack,
    minimal_refutation, pairs_separation, witness_to_keys, keys_to_witness, eval_batch_static,
    CLASS_K, CLASS_T, CLASS_S4, CLASS_S5, ACCUMULATE, FULL_SWEEP, KERNEL_AUTO, KERNEL_SCALAR, KERNEL_SLICED,
    REDUCE_BLOCK, REDUCE_WARP, REDUCE_THREAD, NO_WITNESS,
)
