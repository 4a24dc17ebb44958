"""ORACLE for the fused element-wise programs of soax_expr_compile (NEXT-2) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper's user writes whole-array arithmetic, `soax.posArr(0) = soax.velArr(1) - soax.velArr(2)`,
which its expression templates evaluate element by element in one loop.  This module is the
plain definition of what such a program computes, following the language rules stated in include/soax.h:

  * statements run in order; a later statement sees the values assigned by earlier ones (per particle, and since
    every statement is element-wise, "per particle in order" equals "whole array after whole array", which is what
    is done here: one numpy array operation per arithmetic node, no fusion, no reordering);
  * C typing: float32 op float32 -> float32, anything with a float64 -> float64; named scalars and literals with a
    '.' or an exponent are float64; an integer literal takes the type of the other operand; an assignment rounds to
    the type of the target; `a += b` is `a = (T)(a + b)`;
  * a dim-3 field without index expands the statement over c = 0, 1, 2;
  * integer fields can only be compared, masked with '&' or converted with float()/double();
  * conditions (comparison results) can be joined with '&' and '|' (both operands parenthesised comparisons: '&' and '|'
    bind tighter than comparisons, as in Python); cell(G) is the int32 cell index (i0*G + i1)*G + i2 of the particle on a
    G^3 grid, i_c = trunc(pos_c*G) clamped into [0, G-1] (SURVEY.md 8(c) "BINNING" + the clamp stated in include/soax.h);
  * a MASK program is one condition; its value per particle is a byte, 1 where it holds (mask());
  * nothing is contracted: the only fused multiply-adds are the fma() calls, evaluated with std::fma/std::fmaf
    (oracle.fma); min/max are C's fmin/fmax; wrap(x) = x - floor(x) with a result of exactly 1 mapped to 0 (Q3).

The program text is parsed with Python's own `ast` module (the language is a subset of Python's expression
syntax), so this evaluator shares neither parser nor code generator with the CUDA path.
"""
from __future__ import annotations

import ast
import math

import numpy as np

from . import fma as _fma


class ExprError(ValueError):
    pass


class _IntLit:
    """An integer literal: adapts to the type of the other operand."""

    def __init__(self, v: int):
        self.v = v


def _is_float(x) -> bool:
    return isinstance(x, np.ndarray) and x.dtype in (np.float32, np.float64)


def _is_int(x) -> bool:
    return isinstance(x, _IntLit) or (isinstance(x, np.ndarray) and x.dtype.kind in "iu")


def _promote(a, b):
    """C's usual arithmetic conversions restricted to float/double; integer literals adapt."""
    for x in (a, b):
        if not (_is_float(x) or isinstance(x, _IntLit)):
            raise ExprError("floating-point operands required (convert integer fields with float()/double())")
    dts = [x.dtype for x in (a, b) if _is_float(x)]
    dt = np.float64 if (not dts or np.float64 in dts) else np.float32
    return tuple(_to(x, dt) for x in (a, b)), dt


def _to(x, dt):
    if isinstance(x, _IntLit):
        return np.asarray(x.v, dtype=dt)            # exact for the small integers programs use
    return x.astype(dt, copy=False)                 # IEEE round-to-nearest conversion


def _wrap(x):
    w = x - np.floor(x)
    return np.where(w >= 1, np.zeros_like(w), w)


class _Eval:
    def __init__(self, fields: dict, dims: dict, scalars: dict, n: int):
        self.f, self.dims, self.s, self.n = fields, dims, scalars, n
        self.vec_c = None
        self.vec_dim = 0

    def _full(self, x, dt):
        return np.broadcast_to(_to(x, dt), (self.n,)).astype(dt)

    def field(self, name: str, c):
        if name not in self.f:
            raise ExprError(f"unknown name {name!r}")
        dim = self.dims[name]
        if c is None:
            if dim > 1:
                if self.vec_c is None or dim != self.vec_dim:
                    raise ExprError(f"field {name!r} needs a component index (or the dimension of the vector statement's target)")
                c = self.vec_c
            else:
                c = 0
        if not 0 <= c < dim:
            raise ExprError(f"component {c} outside field {name!r}")
        return name, c

    def ev(self, node):
        v = self._ev(node)
        return np.asarray(v) if isinstance(v, np.generic) else v      # numpy turns 0-d results into scalars: keep arrays

    def _ev(self, node):
        if isinstance(node, ast.Constant):
            if isinstance(node.value, bool) or not isinstance(node.value, (int, float)):
                raise ExprError("only numeric literals")
            return _IntLit(node.value) if isinstance(node.value, int) else np.asarray(node.value, dtype=np.float64)
        if isinstance(node, ast.Name):
            if node.id in self.s:
                return np.asarray(self.s[node.id], dtype=np.float64)
            name, c = self.field(node.id, None)
            return self.f[name][c]
        if isinstance(node, ast.Subscript):
            if not isinstance(node.value, ast.Name) or not isinstance(node.slice, ast.Constant):
                raise ExprError("component index must be an integer literal")
            name, c = self.field(node.value.id, int(node.slice.value))
            return self.f[name][c]
        if isinstance(node, ast.UnaryOp):
            v = self.ev(node.operand)
            if isinstance(node.op, ast.UAdd):
                return v
            if not isinstance(node.op, ast.USub):
                raise ExprError("unsupported unary operator")
            if isinstance(v, _IntLit):
                return _IntLit(-v.v)
            if not _is_float(v):
                raise ExprError("unary '-' needs a floating-point operand")
            return -v
        if isinstance(node, ast.BinOp):
            a, b = self.ev(node.left), self.ev(node.right)
            is_cond = lambda x: isinstance(x, np.ndarray) and x.dtype == bool      # noqa: E731
            if isinstance(node.op, (ast.BitAnd, ast.BitOr)) and is_cond(a) and is_cond(b):
                return np.logical_and(a, b) if isinstance(node.op, ast.BitAnd) else np.logical_or(a, b)
            if isinstance(node.op, ast.BitOr):
                raise ExprError("'|' joins two conditions")
            if isinstance(node.op, ast.BitAnd):
                if not (_is_int(a) and _is_int(b)):
                    raise ExprError("'&' needs integer operands or two conditions")
                dt = next(x.dtype for x in (a, b) if isinstance(x, np.ndarray)) if any(isinstance(x, np.ndarray) for x in (a, b)) else np.int64
                av, bv = (np.asarray(x.v, dtype=dt) if isinstance(x, _IntLit) else x for x in (a, b))
                return np.bitwise_and(av, bv)
            (a, b), dt = _promote(a, b)
            if isinstance(node.op, ast.Add):
                r = a + b
            elif isinstance(node.op, ast.Sub):
                r = a - b
            elif isinstance(node.op, ast.Mult):
                r = a * b
            elif isinstance(node.op, ast.Div):
                with np.errstate(divide="ignore", invalid="ignore"):
                    r = a / b
            else:
                raise ExprError("unsupported operator")
            assert r.dtype == dt
            return r
        if isinstance(node, ast.Compare):
            if len(node.ops) != 1:
                raise ExprError("chained comparisons are not part of the language")
            a, b = self.ev(node.left), self.ev(node.comparators[0])
            if _is_int(a) and _is_int(b):
                av, bv = (np.asarray(x.v) if isinstance(x, _IntLit) else x for x in (a, b))
            else:
                (av, bv), _ = _promote(a, b)
            op = node.ops[0]
            table = {ast.Lt: np.less, ast.LtE: np.less_equal, ast.Gt: np.greater, ast.GtE: np.greater_equal,
                     ast.Eq: np.equal, ast.NotEq: np.not_equal}
            for k, fn in table.items():
                if isinstance(op, k):
                    return fn(av, bv)
            raise ExprError("unsupported comparison")
        if isinstance(node, ast.Call):
            if not isinstance(node.func, ast.Name) or node.keywords:
                raise ExprError("unsupported call")
            if node.func.id == "cell":
                return self.cell(node.args)
            return self.call(node.func.id, [self.ev(a) for a in node.args])
        raise ExprError(f"unsupported syntax: {ast.dump(node)}")

    def cell(self, args):
        """a10: i_c = (int32)(pos_c * G) (exact product, truncation), clamped into the grid; cell = (i0*G + i1)*G + i2."""
        if len(args) != 1 or not isinstance(args[0], ast.Constant) or not isinstance(args[0].value, int) or isinstance(args[0].value, bool):
            raise ExprError("cell(G): G must be an integer literal")
        G = args[0].value
        if G < 1 or G > 64 or G & (G - 1):
            raise ExprError("cell(G): G must be a power of two, 1 <= G <= 64")
        if "pos" not in self.f or self.dims["pos"] != 3 or self.f["pos"][0].dtype != np.float64:
            raise ExprError("cell(G) needs a field pos of three doubles")
        i = [np.clip(np.trunc(self.f["pos"][c] * float(G)), 0, G - 1).astype(np.int32) for c in range(3)]
        return (i[0] * np.int32(G) + i[1]) * np.int32(G) + i[2]

    def call(self, fn: str, a: list):
        r = self._call(fn, a)
        return np.asarray(r) if isinstance(r, np.generic) else r

    def _call(self, fn: str, a: list):
        if fn in ("float", "double"):
            dt = np.float32 if fn == "float" else np.float64
            (x,) = a
            if isinstance(x, np.ndarray) and x.dtype == bool:
                raise ExprError("cannot convert a comparison")
            return _to(x, dt)
        if fn == "select":
            c, x, y = a
            if not (isinstance(c, np.ndarray) and c.dtype == bool):
                raise ExprError("select(cond, a, b): cond must be a comparison")
            (x, y), _ = _promote(x, y)
            return np.where(c, x, y)
        arity = {"fma": 3, "sqrt": 1, "abs": 1, "min": 2, "max": 2, "floor": 1, "wrap": 1}
        if fn not in arity or len(a) != arity[fn]:
            raise ExprError(f"unknown function or wrong argument count: {fn}")
        dts = [x.dtype for x in a if _is_float(x)]
        for x in a:
            if not (_is_float(x) or isinstance(x, _IntLit)):
                raise ExprError(f"{fn}() needs floating-point arguments")
        dt = np.float64 if (not dts or np.float64 in dts) else np.float32
        a = [_to(x, dt) for x in a]
        if fn == "fma":
            return _fma(*[np.ascontiguousarray(self._full(x, dt)) for x in a])
        if fn == "sqrt":
            with np.errstate(invalid="ignore"):
                return np.sqrt(a[0])
        if fn == "abs":
            return np.abs(a[0])
        if fn == "min":
            return np.fmin(a[0], a[1])
        if fn == "max":
            return np.fmax(a[0], a[1])
        if fn == "floor":
            return np.floor(a[0])
        return _wrap(a[0])

    def assign(self, target, op, value_node):
        if isinstance(target, ast.Name):
            name, c = self.field(target.id, None)
        elif isinstance(target, ast.Subscript) and isinstance(target.value, ast.Name) and isinstance(target.slice, ast.Constant):
            name, c = self.field(target.value.id, int(target.slice.value))
        else:
            raise ExprError("assignment target must be a field or field[c]")
        cur = self.f[name][c]
        if cur.dtype not in (np.float32, np.float64):
            raise ExprError("assignment to an integer field is not supported")
        v = self.ev(value_node)
        if isinstance(v, _IntLit):
            v = _to(v, cur.dtype)                   # an integer literal takes the type of the target
        if not (_is_float(v)):
            raise ExprError("the right-hand side must be a floating-point value")
        if op is not None:
            (x, y), _ = _promote(cur, v)
            with np.errstate(divide="ignore", invalid="ignore"):
                v = {ast.Add: np.add, ast.Sub: np.subtract, ast.Mult: np.multiply, ast.Div: np.divide}[type(op)](x, y)
        self.f[name][c] = self._full(v, cur.dtype)


def run(fields: dict, source: str, scalars: dict | None = None) -> dict:
    """fields: name -> (dim, N) ndarray (int32/int64/uint8/float32/float64).  Returns a new dict with the program
    applied once; the input is not modified."""
    scalars = dict(scalars or {})
    n = next(iter(fields.values())).shape[1]
    state = {k: [np.array(v[c]) for c in range(v.shape[0])] for k, v in fields.items()}
    dims = {k: v.shape[0] for k, v in fields.items()}
    try:
        tree = ast.parse(source.strip().rstrip(";"))
    except SyntaxError as e:
        raise ExprError(str(e)) from e
    for stmt in tree.body:
        if isinstance(stmt, ast.Assign):
            if len(stmt.targets) != 1:
                raise ExprError("one target per statement")
            target, op, value = stmt.targets[0], None, stmt.value
        elif isinstance(stmt, ast.AugAssign):
            target, op, value = stmt.target, stmt.op, stmt.value
            if not isinstance(op, (ast.Add, ast.Sub, ast.Mult, ast.Div)):
                raise ExprError("unsupported compound assignment")
        else:
            raise ExprError("only assignments are statements")
        tname = target.id if isinstance(target, ast.Name) else getattr(getattr(target, "value", None), "id", None)
        ev = _Eval(state, dims, scalars, n)
        vector_form = isinstance(target, ast.Name) and tname in dims and dims[tname] > 1
        ev.vec_dim = dims.get(tname, 0)
        for c in (range(dims[tname]) if vector_form else [None]):
            ev.vec_c = c
            ev.assign(target, op, value)
    return {k: np.stack(v) for k, v in state.items()}


def total(fields: dict, expression: str, scalars: dict | None = None) -> float:
    """The reduction programs of soax_expr_compile_sum: the expression is evaluated per particle as in `run`, converted
    to float64, and the terms are added exactly (math.fsum: the correctly rounded sum, so no summation order is implied)."""
    n = next(iter(fields.values())).shape[1]
    state = {k: [np.array(v[c]) for c in range(v.shape[0])] for k, v in fields.items()}
    dims = {k: v.shape[0] for k, v in fields.items()}
    try:
        tree = ast.parse(expression.strip().rstrip(";"), mode="eval")
    except SyntaxError as e:
        raise ExprError(str(e)) from e
    v = _Eval(state, dims, dict(scalars or {}), n).ev(tree.body)
    if isinstance(v, _IntLit):
        v = _to(v, np.float64)
    if not _is_float(v):
        raise ExprError("the summed expression must be a floating-point value")
    terms = np.broadcast_to(v.astype(np.float64), (n,))
    return math.fsum(terms.tolist())


def mask(fields: dict, condition: str, scalars: dict | None = None) -> np.ndarray:
    """The mask programs of soax_expr_compile_mask: one condition, evaluated per particle as in `run`; returns uint8, 1 where
    it holds."""
    n = next(iter(fields.values())).shape[1]
    state = {k: [np.array(v[c]) for c in range(v.shape[0])] for k, v in fields.items()}
    dims = {k: v.shape[0] for k, v in fields.items()}
    try:
        tree = ast.parse(condition.strip().rstrip(";"), mode="eval")
    except SyntaxError as e:
        raise ExprError(str(e)) from e
    v = _Eval(state, dims, dict(scalars or {}), n).ev(tree.body)
    if not (isinstance(v, np.ndarray) and v.dtype == bool):
        raise ExprError("the mask expression must be a condition")
    return np.broadcast_to(v, (n,)).astype(np.uint8)
