"""Seeded synthetic inputs (formula corpora, formula pairs, frame ranges).

This package is the ONLY code shared by the oracle (`oracle/`) and the CUDA path
(`paper_2606_15437_b200/`).  It holds no evaluation arithmetic: it only builds formula
syntax trees, serialises them as postfix bytes (the wire format of `include/kripke.h`)
and draws seeded random numbers.  See DESIGN.md "Input recipe".
"""
from .formulas import (  # noqa: F401
    OP_TOP, OP_BOT, OP_VAR0, OP_NOT, OP_BOX, OP_DIA, OP_AND, OP_OR, OP_IMP,
    parse, to_postfix, from_postfix, to_text, node_count, modal_depth, n_vars_used,
    pack_programs, unpack_programs,
)
from .corpus import (  # noqa: F401
    SplitMix64, gen_formula, corpus_c1, corpus_c2, corpus_c4, pairs_c5,
    enumerate_constant_free, named_axioms, alpha,
)
