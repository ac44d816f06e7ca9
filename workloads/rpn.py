"""Tiny expression builder that emits the postfix (RPN) int32 constraint programs of include/cao.h.

Program words (int32):  PUSH_PARAM d | PUSH_CONST lo hi | binary/unary opcodes.  This module only
*encodes* programs; it never evaluates them (the oracle and the CUDA library each have their own
interpreter, and the tests' brute-force reference uses hand-written Python predicates instead).
"""
from __future__ import annotations

OPCODES = {
    "PUSH_PARAM": 1, "PUSH_CONST": 2,
    "ADD": 3, "SUB": 4, "MUL": 5, "DIV": 6, "MOD": 7, "NEG": 8, "MIN": 9, "MAX": 10,
    "LT": 11, "LE": 12, "GT": 13, "GE": 14, "EQ": 15, "NE": 16,
    "AND": 17, "OR": 18, "NOT": 19,
}


def _wrap(x) -> "Expr":
    if isinstance(x, Expr):
        return x
    if isinstance(x, int):
        return C(x)
    raise TypeError(f"cannot use {type(x)} in a constraint expression")


class Expr:
    """Postfix word list with operator overloading (comparison operators build programs too)."""

    def __init__(self, words):
        self.words = list(words)

    def _bin(self, other, op):
        return Expr(self.words + _wrap(other).words + [OPCODES[op]])

    def _rbin(self, other, op):
        return Expr(_wrap(other).words + self.words + [OPCODES[op]])

    def __add__(self, o): return self._bin(o, "ADD")
    def __radd__(self, o): return self._rbin(o, "ADD")
    def __sub__(self, o): return self._bin(o, "SUB")
    def __rsub__(self, o): return self._rbin(o, "SUB")
    def __mul__(self, o): return self._bin(o, "MUL")
    def __rmul__(self, o): return self._rbin(o, "MUL")
    def __floordiv__(self, o): return self._bin(o, "DIV")      # C semantics: truncates toward zero
    def __rfloordiv__(self, o): return self._rbin(o, "DIV")
    def __mod__(self, o): return self._bin(o, "MOD")           # C semantics: sign of the dividend
    def __rmod__(self, o): return self._rbin(o, "MOD")
    def __neg__(self): return Expr(self.words + [OPCODES["NEG"]])
    def __lt__(self, o): return self._bin(o, "LT")
    def __le__(self, o): return self._bin(o, "LE")
    def __gt__(self, o): return self._bin(o, "GT")
    def __ge__(self, o): return self._bin(o, "GE")
    def eq(self, o): return self._bin(o, "EQ")
    def ne(self, o): return self._bin(o, "NE")

    def program(self):
        return [int(w) for w in self.words]


def P(d: int) -> Expr:
    """Value of parameter (digit) d."""
    return Expr([OPCODES["PUSH_PARAM"], int(d)])


def C(c: int) -> Expr:
    """int64 constant, split into two int32 words (lo, hi)."""
    c = int(c)
    if not -(1 << 63) <= c < (1 << 63):
        raise ValueError("constant out of int64 range")
    u = c & 0xFFFFFFFFFFFFFFFF
    lo, hi = u & 0xFFFFFFFF, u >> 32
    s32 = lambda w: w - (1 << 32) if w >= (1 << 31) else w
    return Expr([OPCODES["PUSH_CONST"], s32(lo), s32(hi)])


def MIN(a, b): return _wrap(a)._bin(b, "MIN")
def MAX(a, b): return _wrap(a)._bin(b, "MAX")
def AND(a, b): return _wrap(a)._bin(b, "AND")
def OR(a, b): return _wrap(a)._bin(b, "OR")
def NOT(a): return Expr(_wrap(a).words + [OPCODES["NOT"]])
