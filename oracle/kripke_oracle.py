"""Tier-1 oracle: Kripke satisfaction written out from the definitions.  TEST INFRASTRUCTURE.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` leg may
import this package.  It shares no code with `paper_2606_15437_b200/` (the CUDA path): it has its
own opcode table, its own postfix decoder and its own semantics, over explicit world lists,
relation sets (sets of pairs) and valuation sets.  There is no bit trick in the semantics; bits
appear only where an integer index (frame f, valuation v) is decoded into those sets.

What it follows:
  * satisfaction, truth set, frame validity, countermodel: PAPER.md:38-42 (section 2);
  * frame classes K / T / S4 / S5 by their first-order definitions: PAPER.md:42;
  * certificate and its checker: PAPER.md:129-135 (Definition 1, Proposition 2);
  * least refuting size: PAPER.md:137-139 (Theorem 2(2));
  * k-indistinguishability as a disagreement world: PAPER.md:169-173 (Def. 2, Prop. 4);
  * index conventions (readings R2, R3): edge w->u is bit (w*n+u) of f, i.e.
    succ[w] = (f >> w*n) & (2^n-1); variable p_i holds at w iff bit (i*n+w) of v.
Pins: tests/test_oracle_pins.py (closed forms, the paper's worked certificate, Lemma 2, ...).
"""
from __future__ import annotations

NO_WITNESS = (1 << 64) - 1

CLASS_K, CLASS_T, CLASS_S4, CLASS_S5 = 0, 1, 2, 3

# own copy of the wire format of include/kripke.h
_TOP, _BOT, _VAR0, _NOT, _BOX, _DIA, _AND, _OR, _IMP = 0x00, 0x01, 0x10, 0x20, 0x21, 0x22, 0x30, 0x31, 0x32


# ---------------------------------------------------------------------------------------------
# syntax
# ---------------------------------------------------------------------------------------------
def parse_postfix(code: bytes):
    """Postfix bytes -> tree of tuples ('top',) ('bot',) ('var', i) (op, a) (op, a, b)."""
    st = []
    for c in bytes(code):
        if c == _TOP:
            st.append(("top",))
        elif c == _BOT:
            st.append(("bot",))
        elif _VAR0 <= c <= _VAR0 + 3:
            st.append(("var", c - _VAR0))
        elif c in (_NOT, _BOX, _DIA):
            a = st.pop()
            st.append(({_NOT: "not", _BOX: "box", _DIA: "dia"}[c], a))
        elif c in (_AND, _OR, _IMP):
            b = st.pop()
            a = st.pop()
            st.append(({_AND: "and", _OR: "or", _IMP: "imp"}[c], a, b))
        else:
            raise ValueError(f"bad opcode 0x{c:02x}")
    if len(st) != 1:
        raise ValueError("malformed postfix program")
    return st[0]


# ---------------------------------------------------------------------------------------------
# models from indices (the only place bits are read)
# ---------------------------------------------------------------------------------------------
def relation_from_index(n: int, f: int):
    """R = {(w, u) : bit (w*n + u) of f is 1}  (reading R2)."""
    return {(w, u) for w in range(n) for u in range(n) if (f >> (w * n + u)) & 1}


def relation_from_succ(n: int, succ):
    """R from successor masks as printed in a certificate (bit u of succ[w])."""
    return {(w, u) for w in range(n) for u in range(n) if (succ[w] >> u) & 1}


def index_from_relation(n: int, R) -> int:
    return sum(1 << (w * n + u) for (w, u) in R)


def valuation_from_index(n: int, k: int, v: int):
    """V(p_i) = {w : bit (i*n + w) of v is 1}  (reading R3)."""
    return [{w for w in range(n) if (v >> (i * n + w)) & 1} for i in range(k)]


# ---------------------------------------------------------------------------------------------
# semantics
# ---------------------------------------------------------------------------------------------
def sat(n, R, V, w, phi) -> bool:
    """M, w |= phi, by recursion on phi.  R is a set of pairs, V a list of sets."""
    tag = phi[0]
    if tag == "top":
        return True
    if tag == "bot":
        return False
    if tag == "var":
        return w in V[phi[1]]
    if tag == "not":
        return not sat(n, R, V, w, phi[1])
    if tag == "and":
        return sat(n, R, V, w, phi[1]) and sat(n, R, V, w, phi[2])
    if tag == "or":
        return sat(n, R, V, w, phi[1]) or sat(n, R, V, w, phi[2])
    if tag == "imp":
        return (not sat(n, R, V, w, phi[1])) or sat(n, R, V, w, phi[2])
    if tag == "box":   # every R-successor satisfies; true at a dead end
        return all(sat(n, R, V, u, phi[1]) for u in range(n) if (w, u) in R)
    if tag == "dia":   # some R-successor satisfies; false at a dead end
        return any(sat(n, R, V, u, phi[1]) for u in range(n) if (w, u) in R)
    raise ValueError(tag)


def truth_set(n, R, V, phi):
    """[[phi]] as the sorted list of worlds."""
    return [w for w in range(n) if sat(n, R, V, w, phi)]


def refutes(n, R, V, phi) -> bool:
    """The model refutes phi iff its truth set is not all of W."""
    return truth_set(n, R, V, phi) != list(range(n))


# ---------------------------------------------------------------------------------------------
# frame classes by first-order definitions
# ---------------------------------------------------------------------------------------------
def is_reflexive(n, R):
    return all((w, w) in R for w in range(n))


def is_transitive(n, R):
    return all((w, t) in R for (w, u) in R for (u2, t) in R if u2 == u)


def is_symmetric(n, R):
    return all((u, w) in R for (w, u) in R)


def in_class(n, R, cls) -> bool:
    if cls == CLASS_K:
        return True
    if cls == CLASS_T:
        return is_reflexive(n, R)
    if cls == CLASS_S4:
        return is_reflexive(n, R) and is_transitive(n, R)
    if cls == CLASS_S5:
        return is_reflexive(n, R) and is_transitive(n, R) and is_symmetric(n, R)
    raise ValueError("bad class")


def class_frames(n, cls):
    """Ascending list of the K-indices f whose relation is in the class (reading R10)."""
    return [f for f in range(1 << (n * n)) if in_class(n, relation_from_index(n, f), cls)]


# ---------------------------------------------------------------------------------------------
# census over a frame range (Algorithm 1's outputs, readings R6, R7, R8)
# ---------------------------------------------------------------------------------------------
def census(code, n, k, cls=CLASS_K, frame_begin=0, frame_count=None, frames=None):
    """One formula over class frames [frame_begin, frame_begin+frame_count) (class order = ascending
    f) and all 2^(k*n) valuations, ascending.

    Returns (refuting_models, refuting_frames, witness) with witness = (f, v, w): the first
    refuting (f, v) in that order and the least world outside the truth set, or
    (NO_WITNESS, 0, 0) if nothing in the range refutes.
    """
    phi = parse_postfix(code)
    if frames is None:
        frames = class_frames(n, cls)
    if frame_count is None:
        frame_count = len(frames) - frame_begin
    models = 0
    nframes = 0
    witness = (NO_WITNESS, 0, 0)
    everything = list(range(n))
    for f in frames[frame_begin:frame_begin + frame_count]:
        R = relation_from_index(n, f)
        hit = False
        for v in range(1 << (k * n)):
            V = valuation_from_index(n, k, v)
            ts = truth_set(n, R, V, phi)
            if ts != everything:
                models += 1
                hit = True
                if witness[0] == NO_WITNESS:
                    witness = (f, v, min(w for w in everything if w not in ts))
        nframes += hit
    return models, nframes, witness


def distinguish(code_a, code_b, n, k, cls=CLASS_K, frame_begin=0, frame_count=None, frames=None):
    """Pair path: a model distinguishes phi, psi iff some world satisfies exactly
    one of them.  Returns (distinguishing_models, distinguishing_frames, (f, v, w)) with w the least
    disagreement world of the first distinguishing (f, v)."""
    phi = parse_postfix(code_a)
    psi = parse_postfix(code_b)
    if frames is None:
        frames = class_frames(n, cls)
    if frame_count is None:
        frame_count = len(frames) - frame_begin
    models = 0
    nframes = 0
    witness = (NO_WITNESS, 0, 0)
    for f in frames[frame_begin:frame_begin + frame_count]:
        R = relation_from_index(n, f)
        hit = False
        for v in range(1 << (k * n)):
            V = valuation_from_index(n, k, v)
            D = [w for w in range(n) if sat(n, R, V, w, phi) != sat(n, R, V, w, psi)]
            if D:
                models += 1
                hit = True
                if witness[0] == NO_WITNESS:
                    witness = (f, v, min(D))
        nframes += hit
    return models, nframes, witness


# ---------------------------------------------------------------------------------------------
# explicit frame lists (PAPER.md:183-185 stress templates, :192 synthesized relations)
# ---------------------------------------------------------------------------------------------
def relation_from_matrix(n: int, mat):
    """R from an n x n 0/1 adjacency matrix: mat[w][u] != 0 iff w -> u."""
    return {(w, u) for w in range(n) for u in range(n) if mat[w][u]}


def census_relations(code, n, k, mats):
    """One formula over an explicit list of frames (adjacency matrices, any n) and all 2^(k*n)
    valuations.  Same outputs as `census`, the witness frame being the POSITION j in the list:
    (refuting_models, refuting_frames, (j, v, w))."""
    phi = parse_postfix(code)
    everything = list(range(n))
    models = nframes = 0
    witness = (NO_WITNESS, 0, 0)
    for j, mat in enumerate(mats):
        R = relation_from_matrix(n, mat)
        hit = False
        for v in range(1 << (k * n)):
            V = valuation_from_index(n, k, v)
            ts = truth_set(n, R, V, phi)
            if ts != everything:
                models += 1
                hit = True
                if witness[0] == NO_WITNESS:
                    witness = (j, v, min(w for w in everything if w not in ts))
        nframes += hit
    return models, nframes, witness


def distinguish_relations(code_a, code_b, n, k, mats):
    """Pair path over an explicit list of frames; witness = (position, v, least
    disagreement world)."""
    phi = parse_postfix(code_a)
    psi = parse_postfix(code_b)
    models = nframes = 0
    witness = (NO_WITNESS, 0, 0)
    for j, mat in enumerate(mats):
        R = relation_from_matrix(n, mat)
        hit = False
        for v in range(1 << (k * n)):
            V = valuation_from_index(n, k, v)
            D = [w for w in range(n) if sat(n, R, V, w, phi) != sat(n, R, V, w, psi)]
            if D:
                models += 1
                hit = True
                if witness[0] == NO_WITNESS:
                    witness = (j, v, min(D))
        nframes += hit
    return models, nframes, witness


# ---------------------------------------------------------------------------------------------
# certificates and least refuting size
# ---------------------------------------------------------------------------------------------
def check_certificate(code, n, succ, val_masks, w, cls) -> bool:
    """Definition 1: valid iff the frame is in the class and M, w does not satisfy phi.
    `succ` are the n successor masks, `val_masks` one world mask per variable."""
    phi = parse_postfix(code)
    R = relation_from_succ(n, succ)
    V = [{u for u in range(n) if (m >> u) & 1} for m in val_masks]
    if not (0 <= w < n):
        return False
    return in_class(n, R, cls) and not sat(n, R, V, w, phi)


def check_witness(code, n, k, cls, f, v, w) -> bool:
    """A census witness (f, v, w) as a certificate."""
    succ = [(f >> (x * n)) & ((1 << n) - 1) for x in range(n)]
    vals = [(v >> (i * n)) & ((1 << n) - 1) for i in range(k)]
    return check_certificate(code, n, succ, vals, w, cls)


def check_pair_witness(code_a, code_b, n, k, cls, f, v, w) -> bool:
    """Proposition 4: the world is one at which phi and psi disagree, on a frame of the class."""
    R = relation_from_index(n, f)
    V = valuation_from_index(n, k, v)
    if not in_class(n, R, cls):
        return False
    return sat(n, R, V, w, parse_postfix(code_a)) != sat(n, R, V, w, parse_postfix(code_b))
