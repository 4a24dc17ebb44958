"""Seeded random expression programs over the wide record R2 (test helper, shared by the CPU compile test and the GPU
parity test of NEXT-2).  The generator only builds program TEXT; it holds none of the language's semantics.  Programs
avoid NaN (sqrt and division are guarded) so that results can be compared bit for bit."""
import random

DOUBLES = [f"{f}[{c}]" for f in ("pos", "vel", "acc") for c in range(3)]
FLOATS = ["mass", "charge"]
TARGETS = DOUBLES + FLOATS


def _leaf(rng):
    r = rng.random()
    if r < 0.45:
        return rng.choice(DOUBLES)
    if r < 0.65:
        return rng.choice(FLOATS)
    if r < 0.75:
        return rng.choice(["double(id)", "float(flags)", "double(flags & 7)"])
    if r < 0.87:
        return rng.choice(["a", "b"])
    return rng.choice(["0.5", "2", "3.25", "1e-3", "7"])


def _expr(rng, depth):
    if depth == 0 or rng.random() < 0.15:
        return _leaf(rng)
    e = lambda: _expr(rng, depth - 1)  # noqa: E731
    kind = rng.randrange(13)
    if kind < 3:
        return f"({e()} {rng.choice('+-*')} {e()})"
    if kind == 3:
        return f"({e()} / (abs({e()}) + 1))"
    if kind == 4:
        return f"fma({e()}, {e()}, {e()})"
    if kind == 5:
        return f"sqrt(abs({e()}))"
    if kind == 6:
        return f"{rng.choice(['abs', 'floor', 'wrap', 'float', 'double'])}({e()})"
    if kind == 7:
        return f"{rng.choice(['min', 'max'])}({e()}, {e()})"
    if kind == 8:
        return f"select({e()} {rng.choice(['<', '<=', '>', '>=', '==', '!='])} {e()}, {e()}, {e()})"
    if kind == 9:
        return f"select((flags & {rng.choice([1, 2, 4, 128])}) != 0, {e()}, {e()})"
    if kind == 10:
        return f"(-{e()})"
    if kind == 11:
        return f"({e()} * 0.25 + {e()})"
    return f"select(double(id) < {rng.choice([10, 1000, 100000])}, {e()}, {e()})"


def program(seed: int) -> str:
    rng = random.Random(seed)
    stmts = []
    for _ in range(rng.randint(1, 4)):
        if rng.random() < 0.2:
            f = rng.choice(["pos", "vel", "acc"])                    # vector form: un-indexed 3-vectors on both sides
            g = rng.choice(["pos", "vel", "acc"])
            stmts.append(f"{f} {rng.choice(['=', '+=', '-=', '*='])} {g} * {_expr(rng, 1)}")
        else:
            op = rng.choice(['=', '=', '+=', '-=', '*=', '/='])
            rhs = _expr(rng, 3)
            stmts.append(f"{rng.choice(TARGETS)} {op} " + (f"(abs({rhs}) + 1)" if op == "/=" else rhs))   # no division by zero
    return "; ".join(stmts)


def _cond(rng, depth):
    """a random condition over R2: comparisons of float expressions, integer tests, cell tests, joined by & and |"""
    if depth > 0 and rng.random() < 0.6:
        return f"({_cond(rng, depth - 1)}) {rng.choice('&|')} ({_cond(rng, depth - 1)})"
    kind = rng.randrange(6)
    if kind < 2:
        return f"{_expr(rng, 2)} {rng.choice(['<', '<=', '>', '>=', '==', '!='])} {_expr(rng, 2)}"
    if kind == 2:
        return f"(flags & {rng.choice([1, 2, 4, 64, 255])}) {rng.choice(['!=', '=='])} {rng.choice([0, 0, 4])}"
    if kind == 3:
        G = rng.choice([1, 2, 8, 64])
        return f"cell({G}) {rng.choice(['<', '>=', '==', '!='])} {rng.randrange(max(1, G ** 3))}"
    if kind == 4:
        G = rng.choice([4, 16, 64])
        return f"double(cell({G})) {rng.choice(['<', '>='])} {rng.choice(['a * 1000', 'lo', '0.5 * lo'])}"
    return f"id {rng.choice(['<', '>=', '!='])} {rng.randrange(600)}"


def condition(seed: int) -> str:
    """one mask program (soax_expr_compile_mask) over R2 with the scalars a, b, lo"""
    return _cond(random.Random(10_000 + seed), 2)
