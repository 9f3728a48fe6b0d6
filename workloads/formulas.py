"""Formula syntax: trees, text, and the postfix byte format.

A formula tree is a nested tuple:
    ("top",) ("bot",) ("var", i) ("not", a) ("box", a) ("dia", a)
    ("and", a, b) ("or", a, b) ("imp", a, b)
Grammar: PAPER.md:38 (section 2).  The postfix byte codes are the wire format declared in
include/kripke.h (the paper gives none; SURVEY.md 8(b) proposal is adopted):
    0x00 top, 0x01 bot, 0x10+i variable p_i, 0x20 not, 0x21 box, 0x22 dia,
    0x30 and, 0x31 or, 0x32 imp (pops y then x, pushes x -> y).
Nothing in this file evaluates a formula.
"""
from __future__ import annotations

import numpy as np

OP_TOP, OP_BOT = 0x00, 0x01
OP_VAR0 = 0x10
OP_NOT, OP_BOX, OP_DIA = 0x20, 0x21, 0x22
OP_AND, OP_OR, OP_IMP = 0x30, 0x31, 0x32

_UNARY = {"not": OP_NOT, "box": OP_BOX, "dia": OP_DIA}
_BINARY = {"and": OP_AND, "or": OP_OR, "imp": OP_IMP}
_UNARY_INV = {v: k for k, v in _UNARY.items()}
_BINARY_INV = {v: k for k, v in _BINARY.items()}
_VAR_NAMES = "pqrs"


def to_postfix(t) -> bytes:
    """Serialise a tree as postfix bytes (iterative; left operand first)."""
    out = bytearray()
    stack = [(t, False)]
    while stack:
        node, done = stack.pop()
        tag = node[0]
        if tag == "top":
            out.append(OP_TOP)
        elif tag == "bot":
            out.append(OP_BOT)
        elif tag == "var":
            out.append(OP_VAR0 + node[1])
        elif done:
            out.append(_UNARY[tag] if tag in _UNARY else _BINARY[tag])
        else:
            stack.append((node, True))
            if tag in _BINARY:
                stack.append((node[2], False))
            stack.append((node[1], False))
    return bytes(out)


def from_postfix(code: bytes):
    """Rebuild the tree from postfix bytes; raises ValueError if malformed."""
    st = []
    for c in code:
        if c == OP_TOP:
            st.append(("top",))
        elif c == OP_BOT:
            st.append(("bot",))
        elif OP_VAR0 <= c < OP_VAR0 + 4:
            st.append(("var", c - OP_VAR0))
        elif c in _UNARY_INV:
            if not st:
                raise ValueError("stack underflow")
            st.append((_UNARY_INV[c], st.pop()))
        elif c in _BINARY_INV:
            if len(st) < 2:
                raise ValueError("stack underflow")
            y = st.pop()
            x = st.pop()
            st.append((_BINARY_INV[c], x, y))
        else:
            raise ValueError(f"bad opcode 0x{c:02x}")
    if len(st) != 1:
        raise ValueError("program does not leave exactly one value")
    return st[0]


def node_count(t) -> int:
    return 1 + sum(node_count(c) for c in t[1:] if isinstance(c, tuple))


def modal_depth(t) -> int:
    d = max((modal_depth(c) for c in t[1:] if isinstance(c, tuple)), default=0)
    return d + (1 if t[0] in ("box", "dia") else 0)


def n_vars_used(t) -> int:
    """1 + the largest variable index mentioned (0 if none)."""
    if t[0] == "var":
        return t[1] + 1
    return max((n_vars_used(c) for c in t[1:] if isinstance(c, tuple)), default=0)


def to_text(t) -> str:
    tag = t[0]
    if tag == "top":
        return "T"
    if tag == "bot":
        return "F"
    if tag == "var":
        return _VAR_NAMES[t[1]]
    if tag == "not":
        return "~" + to_text(t[1])
    if tag == "box":
        return "[]" + to_text(t[1])
    if tag == "dia":
        return "<>" + to_text(t[1])
    sym = {"and": "&", "or": "|", "imp": "->"}[tag]
    return "(" + to_text(t[1]) + sym + to_text(t[2]) + ")"


class _Parser:
    """Text syntax: p q r s, T, F, ~x, []x, <>x, x&y, x|y, x->y (right assoc), parentheses.
    Precedence: unary > & > | > ->."""

    def __init__(self, s: str):
        self.s = s.replace(" ", "")
        self.i = 0

    def peek(self, tok: str) -> bool:
        return self.s.startswith(tok, self.i)

    def eat(self, tok: str) -> bool:
        if self.peek(tok):
            self.i += len(tok)
            return True
        return False

    def imp(self):
        a = self.disj()
        if self.eat("->"):
            return ("imp", a, self.imp())
        return a

    def disj(self):
        a = self.conj()
        while self.eat("|"):
            a = ("or", a, self.conj())
        return a

    def conj(self):
        a = self.unary()
        while self.eat("&"):
            a = ("and", a, self.unary())
        return a

    def unary(self):
        if self.eat("~"):
            return ("not", self.unary())
        if self.eat("[]"):
            return ("box", self.unary())
        if self.eat("<>"):
            return ("dia", self.unary())
        if self.eat("("):
            a = self.imp()
            if not self.eat(")"):
                raise ValueError("expected )")
            return a
        if self.eat("T"):
            return ("top",)
        if self.eat("F"):
            return ("bot",)
        if self.i < len(self.s) and self.s[self.i] in _VAR_NAMES:
            v = _VAR_NAMES.index(self.s[self.i])
            self.i += 1
            return ("var", v)
        raise ValueError(f"parse error at {self.i} in {self.s!r}")


def parse(s: str):
    p = _Parser(s)
    t = p.imp()
    if p.i != len(p.s):
        raise ValueError(f"trailing input at {p.i} in {p.s!r}")
    return t


def pack_programs(programs):
    """List of postfix byte strings -> (code uint8[total], offsets uint32[B+1])."""
    offs = np.zeros(len(programs) + 1, dtype=np.uint32)
    if programs:
        offs[1:] = np.cumsum([len(p) for p in programs], dtype=np.uint64).astype(np.uint32)
    code = np.frombuffer(b"".join(programs), dtype=np.uint8).copy()
    return code, offs


def unpack_programs(code, offsets):
    code = np.asarray(code, dtype=np.uint8)
    return [bytes(code[int(offsets[i]):int(offsets[i + 1])]) for i in range(len(offsets) - 1)]
