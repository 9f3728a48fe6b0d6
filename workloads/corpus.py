"""Seeded formula corpora with the shape of the paper's workloads.

The paper's census corpus (section 6: 5,624 formulas of <= 7 nodes over two
variables) is not in the container; the seeded corpora below stand in for it.  The generator is
SURVEY.md 8(d)'s `gen(budget, depth_left, atoms)`, "uniform over node types".  The PRNG is a
SplitMix64 written out here so the bytes are identical on every machine and Python version.
No evaluation arithmetic lives in this file.
"""
from __future__ import annotations

from .formulas import parse, to_postfix, node_count, modal_depth

_MASK64 = (1 << 64) - 1

SEED_C1 = 15437001
SEED_C2 = 15437002   # also C3: the n=5 census uses the same 5,624-formula file
SEED_C4 = 15437004
SEED_C5 = 15437005


class SplitMix64:
    """Counter-based 64-bit generator (Steele, Lea, Flood 2014), restated."""

    def __init__(self, seed: int):
        self.state = seed & _MASK64

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
        return z ^ (z >> 31)

    def below(self, n: int) -> int:
        """Uniform integer in [0, n) by rejection (no modulo bias)."""
        if n <= 0:
            raise ValueError("n must be positive")
        limit = ((1 << 64) // n) * n
        while True:
            x = self.next_u64()
            if x < limit:
                return x % n


def _atom(name):
    if name == "T":
        return ("top",)
    if name == "F":
        return ("bot",)
    return ("var", "pqrs".index(name))


def gen_formula(rng: SplitMix64, budget: int, depth_left: int, atoms: str):
    """One random formula of at most `budget` nodes and modal depth at most `depth_left`.

    Allowed node types at a call: ATOM always; NOT if budget >= 2; BOX, DIA if budget >= 2 and
    depth_left >= 1; AND, OR, IMP if budget >= 3.  One is picked uniformly among the allowed.
    """
    kinds = ["atom"]
    if budget >= 2:
        kinds.append("not")
        if depth_left >= 1:
            kinds += ["box", "dia"]
    if budget >= 3:
        kinds += ["and", "or", "imp"]
    kind = kinds[rng.below(len(kinds))]
    if kind == "atom":
        return _atom(atoms[rng.below(len(atoms))])
    if kind == "not":
        return ("not", gen_formula(rng, budget - 1, depth_left, atoms))
    if kind in ("box", "dia"):
        return (kind, gen_formula(rng, budget - 1, depth_left - 1, atoms))
    left_budget = 1 + rng.below(budget - 2)
    left = gen_formula(rng, left_budget, depth_left, atoms)
    right = gen_formula(rng, budget - 1 - node_count(left), depth_left, atoms)
    return (kind, left, right)


def _distinct(rng, count, budget, depth, atoms, keep=lambda t: True):
    seen = set()
    out = []
    while len(out) < count:
        t = gen_formula(rng, budget, depth, atoms)
        if not keep(t):
            continue
        code = to_postfix(t)
        if code in seen:
            continue
        seen.add(code)
        out.append(code)
    return out


def corpus_c1(count: int = 1000, seed: int = SEED_C1):
    """Config 1: distinct formulas of <= 7 nodes over atoms {p, q, T, F}; postfix byte strings."""
    return _distinct(SplitMix64(seed), count, 7, 7, "pqTF")


def corpus_c2(count: int = 5624, seed: int = SEED_C2):
    """Configs 2 and 3: 5,624 distinct formulas of <= 7 nodes, modal depth <= 3, atoms {p,q,T,F}."""
    return _distinct(SplitMix64(seed), count, 7, 3, "pqTF")


def corpus_c4(count: int = 2048, seed: int = SEED_C4):
    """Config 4: distinct formulas over {p,q,r} with 9..15 nodes and modal depth 1..6."""
    def keep(t):
        return 9 <= node_count(t) <= 15 and 1 <= modal_depth(t) <= 6
    return _distinct(SplitMix64(seed), count, 15, 6, "pqr", keep)


def alpha(m: int):
    """alpha_m = ([]<>)^m T  (Proposition 5)."""
    t = ("top",)
    for _ in range(m):
        t = ("box", ("dia", t))
    return t


def _iterate(ctx: str, m: int, base):
    """C^m b for a modal context word such as '[]<>'."""
    ops = []
    i = 0
    while i < len(ctx):
        ops.append("box" if ctx[i:i + 2] == "[]" else "dia")
        i += 2
    t = base
    for _ in range(m):
        for op in reversed(ops):
            t = (op, t)
    return t


def pairs_c5(count: int = 4096, seed: int = SEED_C5):
    """Config 5: variable-free formula pairs.

    Returns (programs, pairs, names): postfix byte strings, a list of (i, j) indices into them,
    and a name per pair ('' for seeded pairs).  Named pairs first: (alpha_m, alpha_{m+1}) m=1,2;
    the 32 pairs (C^m b, C^{m+1} b) of PAPER.md:179; <>^5 T / <>^6 T and []^5 F / []^6 F
    (PAPER.md:190).  Then `count` seeded pairs of two distinct gen(9, 9, {T, F}) formulas.
    """
    programs, index = [], {}

    def add(t):
        code = to_postfix(t)
        if code not in index:
            index[code] = len(programs)
            programs.append(code)
        return index[code]

    pairs, names = [], []
    for m in (1, 2):
        pairs.append((add(alpha(m)), add(alpha(m + 1))))
        names.append(f"alpha_{m}/alpha_{m + 1}")
    for ctx in ("[]<>", "<>[]", "[][]", "<><>"):
        for base, bname in ((("top",), "T"), (("bot",), "F")):
            for m in range(1, 5):
                pairs.append((add(_iterate(ctx, m, base)), add(_iterate(ctx, m + 1, base))))
                names.append(f"({ctx})^{m}{bname}/({ctx})^{m + 1}{bname}")
    pairs.append((add(_iterate("<>", 5, ("top",))), add(_iterate("<>", 6, ("top",)))))
    names.append("<>^5T/<>^6T")
    pairs.append((add(_iterate("[]", 5, ("bot",))), add(_iterate("[]", 6, ("bot",)))))
    names.append("[]^5F/[]^6F")
    rng = SplitMix64(seed)
    seen = set()
    while len(seen) < count:
        a = to_postfix(gen_formula(rng, 9, 9, "TF"))
        b = to_postfix(gen_formula(rng, 9, 9, "TF"))
        if a == b or (a, b) in seen:
            continue
        seen.add((a, b))
        pairs.append((add(from_code(a)), add(from_code(b))))
        names.append("")
    return programs, pairs, names


def from_code(code: bytes):
    from .formulas import from_postfix
    return from_postfix(code)


def enumerate_constant_free(max_nodes: int = 7, n_vars: int = 2):
    """Every constant-free formula of <= max_nodes nodes over n_vars variables, by node count
    then construction order (44,678 of them for 7 nodes and two variables)."""
    by_size = {1: [("var", i) for i in range(n_vars)]}
    for k in range(2, max_nodes + 1):
        cur = []
        for op in ("not", "box", "dia"):
            cur += [(op, a) for a in by_size[k - 1]]
        for op in ("and", "or", "imp"):
            for i in range(1, k - 1):
                for a in by_size[i]:
                    for b in by_size[k - 1 - i]:
                        cur.append((op, a, b))
        by_size[k] = cur
    out = []
    for k in range(1, max_nodes + 1):
        out += by_size[k]
    return out


def named_axioms():
    """Axioms of PAPER.md Table 9 plus K, as name -> tree."""
    text = {
        "T": "[]p->p", "D": "[]p-><>p", "4": "[]p->[][]p", "5": "<>p->[]<>p",
        "B": "p->[]<>p", "CD": "<>p->[]p", "C4": "[][]p->[]p", "G": "<>[]p->[]<>p",
        "M": "[]<>p-><>[]p", "K": "[](p->q)->([]p->[]q)",
    }
    return {k: parse(v) for k, v in text.items()}
