"""CPU tests of NEXT-2 (fused element-wise programs): the expression ORACLE
(oracle/expr.py) pinned by things other than itself -- the already pinned step oracles, exact rational arithmetic
with one explicit IEEE rounding per operation (tests/exact.py), hand values -- and the host side of the product's
compiler (soax_expr_compile needs NVRTC but no GPU): syntax/type errors, generated code shape, traffic accounting.
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
from oracle import expr as oexpr
from paper_1710_03462_b200 import inputs
from tests.exact import F, rn32, rn64, to_f32, to_f64, wrap_exact

DT = 1e-3
SE = "vel = fma(float(dt), float(-(k*(pos - 0.5))), vel); pos = wrap(fma(dt, double(vel), pos))"


def bits(a):
    a = np.ascontiguousarray(a)
    return a.view({4: np.uint32, 8: np.uint64, 1: np.uint8}[a.dtype.itemsize])


# ------------------------------------------------------------------------------------------- oracle pins
def test_program_reproduces_the_pinned_step_oracles_bit_for_bit():
    h = inputs.make_r1(4099, seed=3)
    h["vel"] *= 40.0                                                 # many particles cross a face
    cur = h
    for _ in range(5):
        cur = oexpr.run(cur, SE, {"dt": DT, "k": 1.0})
    ref = oracle.symplectic_euler(h, DT, 5)
    assert np.array_equal(bits(cur["pos"]), bits(ref["pos"])) and np.array_equal(bits(cur["vel"]), bits(ref["vel"]))
    assert np.array_equal(cur["id"], h["id"])
    d = oexpr.run(h, "pos = wrap(fma(dt, double(vel), pos))", {"dt": DT})
    assert np.array_equal(bits(d["pos"]), bits(oracle.drift(h, DT, 1)["pos"]))


def test_eq1_on_the_papers_float_record():
    """PAPER.md:136 Eq. 1 on Listing 4's all-float record: one float fma per component (Q2, Q19)."""
    rng = np.random.default_rng(0)
    pos, vel = rng.random((3, 777), np.float32), rng.standard_normal((3, 777)).astype(np.float32)
    out = oexpr.run({"pos": pos, "vel": vel}, "pos = fma(float(dt), vel, pos)", {"dt": DT})
    ref_pos, _ = oracle.b6_euler(pos, vel, 0, DT, 1)
    assert np.array_equal(bits(out["pos"]), bits(ref_pos))


def test_each_operation_rounds_once_exact_rational():
    """Every arithmetic node is ONE IEEE operation in the promoted type: restated with exact rationals."""
    rng = np.random.default_rng(1)
    n = 200
    f = {"pos": rng.random((3, n)) * 3 - 1, "vel": rng.standard_normal((3, n)).astype(np.float32)}
    dt = 0.1
    # float - float stays float; product with a double scalar is a double product of the converted float, then a double add
    out = oexpr.run(f, "vel[0] = vel[1] - vel[2]; pos[0] = pos[0] + vel[1]*dt; pos[1] = fma(dt, double(vel[1]), pos[1]);"
                       "pos[2] = wrap(pos[2]); vel[1] = float(pos[1]) * vel[1]; vel[2] /= 3", {"dt": dt})
    contracted_differs = 0
    for i in range(n):
        v1, v2 = F(f["vel"][1, i]), F(f["vel"][2, i])
        assert out["vel"][0, i] == to_f32(rn32(v1 - v2))
        two_roundings = rn64(F(f["pos"][0, i]) + rn64(v1 * F(dt)))
        assert out["pos"][0, i] == to_f64(two_roundings)
        fused = rn64(F(f["pos"][1, i]) + v1 * F(dt))
        assert out["pos"][1, i] == to_f64(fused)
        contracted_differs += rn64(F(f["pos"][0, i]) + v1 * F(dt)) != two_roundings
        assert out["pos"][2, i] == to_f64(wrap_exact(F(f["pos"][2, i])))
        assert out["vel"][1, i] == to_f32(rn32(rn32(fused) * v1))                    # float(pos[1]) sees the NEW pos[1]
        assert out["vel"][2, i] == to_f32(rn32(v2 / 3))                              # integer literal takes the float type
    assert contracted_differs > 0                                    # the pin can tell a contracted product from a plain one


def test_hand_values_sequencing_vector_form_and_masks():
    f = {"id": np.array([[7, 8, 9, 10]], np.int32), "pos": np.array([[.5, .25, 1.5, -0.25]] * 3),
         "vel": np.array([[1, 2, 3, 4], [10, 20, 30, 40], [0, 0, 0, 0]], np.float32),
         "flags": np.array([[1, 2, 3, 0]], np.uint8)}
    out = oexpr.run(f, "pos[0] = vel[1] - vel[0]")                                   # PAPER.md:294's example shape
    assert out["pos"][0].tolist() == [9, 18, 27, 36] and out["pos"][1].tolist() == f["pos"][1].tolist()
    out = oexpr.run(f, "vel += 1; pos = vel")                                        # vector form; later statements see earlier ones
    assert out["pos"].tolist() == [[2, 3, 4, 5], [11, 21, 31, 41], [1, 1, 1, 1]]
    out = oexpr.run(f, "vel[2] = select((flags & 1) != 0, vel[0], -vel[1]); pos[2] = wrap(pos[2]);"
                       "pos[1] = select(double(id) >= 9, max(pos[1], 1), min(pos[1], 0)); vel[0] = sqrt(abs(vel[0] - 5)) * 2")
    assert out["vel"][2].tolist() == [1, -20, 3, -40]
    assert out["pos"][2].tolist() == [.5, .25, .5, .75]
    assert out["pos"][1].tolist() == [0, 0, 1.5, 1]
    assert out["vel"][0].tolist() == [4, np.float32(np.sqrt(np.float32(3))) * 2, np.float32(np.sqrt(np.float32(2))) * 2, 2]
    assert np.array_equal(out["id"], f["id"]) and np.array_equal(out["flags"], f["flags"])
    assert oexpr.run(f, "pos[0] = wrap(-1e-20 * pos[0] * 0 - 1e-20)")["pos"][0].tolist() == [0, 0, 0, 0]   # Q3: -tiny wraps to 0, not 1


@pytest.mark.parametrize("bad", ["pos[3] = 1.0", "pos = id", "foo = 1.0", "id = 1.0", "pos[0] = select(vel[0], 1, 2)",
                                 "pos[0] = vel", "pos[0] = flags + 1.0", "pos[0] = frob(1.0)", "pos = five"])
def test_oracle_rejects_what_the_language_rejects(bad):
    f = {"id": np.zeros((1, 2), np.int32), "pos": np.zeros((3, 2)), "vel": np.zeros((3, 2), np.float32),
         "flags": np.zeros((1, 2), np.uint8), "five": np.zeros((5, 2))}
    with pytest.raises(oexpr.ExprError):
        oexpr.run(f, bad)


# ------------------------------------------------------------------------- host side of the product's compiler
@pytest.fixture(scope="module")
def compiler():
    from paper_1710_03462_b200 import binding as B, container as Cn
    try:
        e = B.soax_expr_compile(B.soax_layout_define(Cn.R1), "pos[0] = pos[0]", [])
    except B.SoaxError as err:
        if err.status == B.SOAX_ERR_UNSUPPORTED:
            pytest.skip("NVRTC is not installed on this machine")
        raise
    B.soax_expr_free(e)
    return B, Cn


def test_compile_generates_one_fused_kernel(compiler):
    B, Cn = compiler
    L = B.soax_layout_define(Cn.R1)
    e = B.soax_expr_compile(L, SE, ["dt", "k"])
    src = B.soax_expr_cuda_source(e)
    assert src.count("__global__") == 1                              # the whole program is ONE kernel (loop fusion)
    assert src.count("= ld_vec<") == 6 and src.count("    st_vec<") == 6   # every array loaded once and stored once
    assert "a.p[0]" not in src                                       # id is never touched: unused fields cost nothing
    assert B.soax_expr_traffic(e) == (36, 36)                        # 72 B/particle, as the hand-written kernel
    B.soax_expr_free(e)
    e = B.soax_expr_compile(L, "pos[0] = vel[1] - vel[2]", [])       # PAPER.md:294; pos[0] is overwritten: not loaded
    assert B.soax_expr_traffic(e) == (8, 8)
    assert B.soax_expr_cuda_source(e).count("= ld_vec<") == 2
    B.soax_expr_free(e)
    e = B.soax_expr_compile(B.soax_layout_define(Cn.R2), "acc = select((flags & 1) != 0, -(k / double(mass)) * (pos - 0.5), acc)", ["k"])
    assert B.soax_expr_traffic(e) == (1 + 4 + 24 + 24, 24)
    B.soax_expr_free(e)


@pytest.mark.parametrize("bad,msg", [("pos[3] = 1.0", "outside field 'pos'"), ("pos = id", "floating-point"), ("foo = 1.0", "unknown field"),
                                     ("id = 1.0", "integer field"), ("pos[0] = select(vel[0], 1, 2)", "comparison"),
                                     ("pos[0] = vel", "components"), ("pos[0] = flags + 1.0", "unknown name"),
                                     ("pos[0] = frob(1.0)", "unknown function"), ("pos[0] = vel[1] -", "expected a value"),
                                     ("pos[0] = 1.0 pos[1] = 2.0", "';'"), ("pos[0] = dt", "unknown name"), ("", "assigns nothing"),
                                     ("pos[0] = fma(1.0, 2.0)", "takes 3"), ("pos[0] = 1.0 $ 2", "unexpected character")])
def test_compile_errors_carry_a_message(compiler, bad, msg):
    B, Cn = compiler
    with pytest.raises(B.SoaxError) as ei:
        B.soax_expr_compile(B.soax_layout_define(Cn.R1), bad, [])
    assert ei.value.status == B.SOAX_ERR_INVALID_ARG and msg in str(ei.value)
    assert msg in B.soax_expr_error()


def test_compile_argument_checks(compiler):
    B, Cn = compiler
    L = B.soax_layout_define(Cn.R1)
    with pytest.raises(B.SoaxError):
        B.soax_expr_compile(L, "pos[0] = pos", ["pos"])              # a scalar may not shadow a field
    with pytest.raises(B.SoaxError):
        B.soax_expr_compile(L, "pos[0] = 1.0", [f"s{i}" for i in range(17)])
    assert B.lib().soax_expr_compile(None, b"x", None, 0, None) == B.SOAX_ERR_INVALID_ARG
    assert B.lib().soax_expr_free(None) == B.SOAX_ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------- run-time layouts
MY_FIELDS = None


def my_fields(B):
    return (("tag", B.SOAX_I64, 1), ("x", B.SOAX_F64, 2), ("temperature", B.SOAX_F32, 1), ("w", B.SOAX_F64, 5), ("alive", B.SOAX_U8, 1))


def test_dynamic_layout_descriptor_and_program(compiler):
    """the container is generic over any attribute list.  A field list that matches no compiled
    instantiation becomes a run-time layout: container + expression programs work, compiled kernel families do not."""
    B, Cn = compiler
    f = my_fields(B)
    L = B.soax_layout_define_dynamic(f)
    assert L == B.soax_layout_define_dynamic(f)                      # identical list -> same handle
    assert B.soax_layout_define_dynamic(Cn.R1) == B.soax_layout_define(Cn.R1)   # a compiled instantiation wins
    with pytest.raises(B.SoaxError) as ei:
        B.soax_layout_define(f)
    assert ei.value.status == B.SOAX_ERR_UNKNOWN_LAYOUT               # the strict call still only knows compiled layouts
    assert B.soax_layout_nfields(L) == 5 and B.soax_layout_ncomp(L) == 10
    assert [B.soax_layout_comp(L, c) for c in (0, 2, 3, 8, 9)] == [(0, 0, B.SOAX_I64), (1, 1, B.SOAX_F64), (2, 0, B.SOAX_F32),
                                                                   (3, 4, B.SOAX_F64), (4, 0, B.SOAX_U8)]
    stride, offs = B.soax_layout_aos(L, True)
    assert stride == 8 + 16 + 4 + 40 + 1 and offs == [0, 8, 16, 24, 28, 36, 44, 52, 60, 68]
    assert B.soax_slab_bytes(L, 1000) == 8192 + 2 * 8192 + 4096 + 5 * 8192 + 1024
    h = B.soax_alloc(L, 10, 1000, 256 * 4096, B.soax_slab_bytes(L, 1000))      # fake device pointer: never dereferenced
    assert B.soax_field_ptr(h, 3, 4) - B.soax_field_ptr(h, 0, 0) == 8192 + 2 * 8192 + 4096 + 4 * 8192
    with pytest.raises(B.SoaxError) as ei:
        B.soax_step(h, B.step_params(B.SOAX_STEP_DRIFT, 1e-3), 1)
    assert ei.value.status == B.SOAX_ERR_UNSUPPORTED
    assert B.soax_scratch_bytes(L, 1000, 8) == 0
    B.soax_free(h)
    e = B.soax_expr_compile(L, "w[4] = select(alive != 0, w[0] * double(temperature) + x[1], w[4]); x = x * 2", [])
    assert B.soax_expr_traffic(e) == (1 + 8 + 4 + 8 + 8 + 8, 8 + 16)
    B.soax_expr_free(e)
    with pytest.raises(B.SoaxError) as ei:
        B.soax_expr_compile(L, "x = w", [])                          # a 5-vector in a 2-vector statement
    assert "different dimension" in str(ei.value)
    for bad in ([("a b", B.SOAX_F32, 1), ("c", B.SOAX_F32, 1)], [("a", B.SOAX_F32, 1), ("a", B.SOAX_F64, 1)], [("a", B.SOAX_F32, 49)]):
        with pytest.raises(B.SoaxError) as ei:
            B.soax_layout_define_dynamic(bad)
        assert ei.value.status == B.SOAX_ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------- reductions
KE = "0.5 * fma(double(vel[2]), double(vel[2]), fma(double(vel[1]), double(vel[1]), double(vel[0]) * double(vel[0])))"
KE_PE = ("0.5 * fma(k*(pos[2]-c), pos[2]-c, fma(k*(pos[1]-c), pos[1]-c, fma(k*(pos[0]-c), pos[0]-c, "
         "fma(double(vel[2]), double(vel[2]), fma(double(vel[1]), double(vel[1]), double(vel[0]) * double(vel[0]))))))")


def test_sum_oracle_against_the_pinned_energy_and_the_hand_fixture():
    """tests/golden/energy_4particles.txt: KE 18.5, total 18.8125 (all dyadic: exact in any order)."""
    vel = np.array([[1, 2, 2], [0, 0, 0], [3, 4, 0], [-1, -1, -1]], np.float32).T.copy()
    pos = np.array([[.5, .5, .5], [0, .5, .5], [.25, .75, .5], [.5, .5, 0]], np.float64).T.copy()
    f = {"id": np.arange(4, dtype=np.int32)[None], "pos": pos, "vel": vel}
    assert oexpr.total(f, KE) == 18.5 and oexpr.total(f, KE_PE, {"k": 1.0, "c": 0.5}) == 18.8125
    h = inputs.make_r1(50000, seed=8)
    for src, kind in ((KE, oracle.KINETIC), (KE_PE, oracle.KINETIC_PLUS_HARMONIC)):
        a, b = oexpr.total(h, src, {"k": 1.0, "c": 0.5}), oracle.energy(h, kind)
        assert abs(a - b) <= 1e-13 * abs(b)                          # exact sum vs the oracle's compensated sum
    assert oexpr.total(h, "1") == 50000.0 and oexpr.total(h, "double(id)") == 50000 * 49999 / 2
    with pytest.raises(oexpr.ExprError):
        oexpr.total(h, "id")


def test_sum_program_compiles_to_one_reduction_kernel(compiler):
    B, Cn = compiler
    L = B.soax_layout_define(Cn.R1)
    e = B.soax_expr_compile_sum(L, KE, [])
    src = B.soax_expr_cuda_source(e)
    assert src.count("__global__") == 1 and "partial[blockIdx.x]" in src and "st_vec<" not in src.split("struct Args")[1]
    assert B.soax_expr_traffic(e) == (12, 0)                         # reads vel only: 12 B/particle, as the hand KE reduction
    B.soax_expr_free(e)
    for bad, msg in (("vel[0] = 1.0", "single expression"), ("id", "floating-point"), ("vel", "components"), ("pos[0] pos[1]", "single expression")):
        with pytest.raises(B.SoaxError) as ei:
            B.soax_expr_compile_sum(L, bad, [])
        assert msg in str(ei.value), (bad, str(ei.value))


def test_random_programs_compile_and_the_oracle_evaluates_them(compiler):
    """60 seeded random programs (tests/random_programs.py): the product's compiler accepts every one of them, its traffic
    accounting matches what the program text touches, and the oracle evaluates them without NaN (the GPU parity test
    compares the same programs bit for bit)."""
    from tests.random_programs import program
    B, Cn = compiler
    L = B.soax_layout_define(Cn.R2)
    host = inputs.make_r2(513, seed=21)
    for seed in range(60):
        src = program(seed)
        e = B.soax_expr_compile(L, src, ["a", "b"])
        r, w = B.soax_expr_traffic(e)
        assert w > 0 and r >= 0
        B.soax_expr_free(e)
        if seed < 20:
            out = oexpr.run(host, src, {"a": 0.75, "b": -1.5})
            assert all(np.isfinite(out[k]).all() for k in ("pos", "vel", "acc", "mass", "charge")), src


# ------------------------------------------------------------------------------------------- masks (NEXT-3 feed)
def test_mask_oracle_hand_values_cell_and_joins(golden_dir):
    """Pins for oexpr.mask / cell() / '&' '|' on conditions: the 6-particle binning fixture (cells 4,1,4,3,1,7
    on a 2^3 grid), the already pinned cell index of oracle.bin_r1 on random positions, hand-written flag tests, and the
    clamp of cell() for a position outside the box."""
    pos = np.array([[.75, .25, .25], [.25, .25, .75], [.75, .25, .40], [.10, .90, .90], [.25, .25, .60], [.99, .99, .99]]).T.copy()
    f = {"id": np.arange(6, dtype=np.int32)[None], "pos": pos, "vel": np.zeros((3, 6), np.float32)}
    assert oexpr.mask(f, "cell(2) == 4").tolist() == [1, 0, 1, 0, 0, 0]
    assert oexpr.mask(f, "(cell(2) < 2) | (cell(2) >= 7)").tolist() == [0, 1, 0, 0, 1, 1]
    assert oexpr.mask(f, "(cell(2) >= 2) & (cell(2) < 7)").tolist() == [1, 0, 1, 1, 0, 0]
    assert oexpr.mask(f, "(double(cell(2)) < lo) | (double(cell(2)) >= hi)", {"lo": 2, "hi": 7}).tolist() == [0, 1, 0, 0, 1, 1]
    assert oexpr.mask(f, "cell(1) == 0").tolist() == [1] * 6
    assert oexpr.mask(f, "(pos[0] > 0.5) & (id != 5)").tolist() == [1, 0, 1, 0, 0, 0]
    assert oexpr.mask(f, "((pos[0] > 0.5) & (id != 5)) | (id == 1)").tolist() == [1, 1, 1, 0, 0, 0]
    h = inputs.make_r1(20000, seed=5)
    for G in (1, 2, 8, 64):
        cell = oracle.bin_r1(h, G, want_perm=False)["cell"]            # pinned by the fixture + brute force in test_oracle_pins
        for k in (0, G ** 3 // 2, G ** 3 - 1):
            assert np.array_equal(oexpr.mask(h, f"cell({G}) == {k}"), (cell == k).astype(np.uint8))
            assert np.array_equal(oexpr.mask(h, f"double(cell({G})) >= t", {"t": k}), (cell >= k).astype(np.uint8))
    out = {"id": np.zeros((1, 3), np.int32), "pos": np.array([[-0.25, 0.5, 1.5], [0.5, 0.5, 0.5], [0.5, 0.5, 0.5]]), "vel": np.zeros((3, 3), np.float32)}
    assert [int(m) for m in (oexpr.mask(out, "cell(4) == 10"), oexpr.mask(out, "cell(4) == 42"), oexpr.mask(out, "cell(4) == 58"))[0:1][0]] == [1, 0, 0]
    assert oexpr.mask(out, "cell(4) == 42").tolist() == [0, 1, 0] and oexpr.mask(out, "cell(4) == 58").tolist() == [0, 0, 1]   # clamped to i0 = 0 / 3
    r2 = inputs.make_r2(1000, seed=2)
    assert np.array_equal(oexpr.mask(r2, "(flags & 1) != 0"), (r2["flags"][0] & 1).astype(np.uint8))
    assert np.array_equal(oexpr.mask(r2, "((flags & 6) == 6) | (mass < 1)"),
                          (((r2["flags"][0] & 6) == 6) | (r2["mass"][0] < np.float32(1))).astype(np.uint8))
    for bad in ("pos[0]", "flags & 1", "(pos[0] < 1) | 3", "cell(3) == 0", "cell(pos) == 0", "(pos[0] < 1) < 2"):
        with pytest.raises(oexpr.ExprError):
            oexpr.mask(r2, bad)


def test_mask_program_compiles_and_rejects(compiler):
    from tests.random_programs import condition
    B, Cn = compiler
    L1, L2 = B.soax_layout_define(Cn.R1), B.soax_layout_define(Cn.R2)
    e = B.soax_expr_compile_mask(L1, "(double(cell(64)) < lo) | (double(cell(64)) >= hi)", ["lo", "hi"])
    src = B.soax_expr_cuda_source(e)
    assert src.count("__global__") == 1 and "soax_cell(" in src and "st_vec<" not in src.split("struct Args")[1]
    assert B.soax_expr_traffic(e) == (24, 1)                          # reads pos only, writes one byte per particle
    B.soax_expr_free(e)
    e = B.soax_expr_compile_mask(L2, "(flags & 1) != 0", [])
    assert B.soax_expr_traffic(e) == (1, 1)
    B.soax_expr_free(e)
    B.soax_expr_free(B.soax_expr_compile_mask(L2, "flags & 1 != 0", []))   # '&' binds tighter than '!=' (Python's rule): (flags & 1) != 0
    assert np.array_equal(oexpr.mask(inputs.make_r2(100, seed=1), "flags & 1 != 0"), oexpr.mask(inputs.make_r2(100, seed=1), "(flags & 1) != 0"))
    for bad, msg in (("pos[0]", "must be a condition"), ("(pos[0] < 1) | 3", "joins two conditions"),
                     ("cell(3) == 1", "power of two"), ("pos[0] < 1; pos[1] < 2", "single condition"), ("vel[0] = 1.0", "")):
        with pytest.raises(B.SoaxError) as ei:
            B.soax_expr_compile_mask(L2, bad, [])
        assert ei.value.status == B.SOAX_ERR_INVALID_ARG and msg in str(ei.value), (bad, str(ei.value))
    with pytest.raises(B.SoaxError):
        B.soax_expr_compile_mask(B.soax_layout_define(Cn.B6(0)), "cell(8) == 0", [])     # pos is float there: no cell()
    with pytest.raises(B.SoaxError):
        B.soax_expr_compile(L2, "mass = 1.0", ["not an identifier"])
    host = inputs.make_r2(777, seed=4)
    for seed in range(24):                                            # the first of the random conditions of the GPU parity test
        src = condition(seed)
        B.soax_expr_free(B.soax_expr_compile_mask(L2, src, ["a", "b", "lo"]))
        m = oexpr.mask(host, src, {"a": 0.75, "b": -1.5, "lo": 3000.0})
        assert m.dtype == np.uint8 and set(np.unique(m)) <= {0, 1}
