"""Pins for the oracle (oracle/soax_oracle.cpp): what the paper and the mathematics fix, never the oracle
itself.  CPU only.  Pin table: SURVEY.md section 8(c) "What pins each part".

Three kinds of pin, chosen so that a dropped term, a wrong sign or index, a swapped operand, a missing
fusion (fma vs mul+add) or a wrong operation order fails at least one:
  * closed forms / invariants of the maps (constant-velocity drift, the linear symplectic-Euler and RK2
    maps, the exact RK2 energy growth factor, the kick-drift invariant);
  * hand fixtures under tests/golden/ (dyadic 4-particle energy, 6-particle binning);
  * exact rational arithmetic with one explicit IEEE rounding per operation (tests/exact.py) and
    O(N^2) brute force on tiny inputs, compared BIT FOR BIT.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1710_03462_b200 import inputs
from tests.exact import F, rn32, rn64, to_f32, to_f64, wrap_exact

DT = 1e-3


def bits(a):
    a = np.ascontiguousarray(a)
    return a.view({4: np.uint32, 8: np.uint64, 1: np.uint8}[a.dtype.itemsize])


def pdist(a, b):
    d = np.abs(np.asarray(a, np.float64) - np.asarray(b, np.float64))
    return np.minimum(d, 1.0 - d)


def r1(pos, vel, ids=None):
    pos = np.asarray(pos, np.float64).reshape(-1, 3)
    vel = np.asarray(vel, np.float32).reshape(-1, 3)
    n = pos.shape[0]
    ids = np.arange(n, dtype=np.int32) if ids is None else np.asarray(ids, np.int32)
    return {"id": ids[None, :].copy(), "pos": np.ascontiguousarray(pos.T), "vel": np.ascontiguousarray(vel.T)}


# ---------------------------------------------------------------------------------------- wrap (a3, Q3)
def test_wrap_special_values():
    assert oracle.wrap(-1e-20) == 0.0                       # x - floor(x) == 1.0 in binary64 -> 0.0
    assert oracle.wrap(1.0) == 0.0 and oracle.wrap(2.0) == 0.0 and oracle.wrap(-1.0) == 0.0
    assert oracle.wrap(0.0) == 0.0 and math.copysign(1.0, oracle.wrap(-0.0)) == 1.0
    top = 1.0 - 2.0 ** -53
    assert oracle.wrap(top) == top
    assert oracle.wrap(1.25) == 0.25 and oracle.wrap(-0.25) == 0.75 and oracle.wrap(-2.5) == 0.5
    assert oracle.wrap(5e-324) == 5e-324 and oracle.wrap(-5e-324) == 0.0


def test_wrap_properties_random():
    rng = np.random.default_rng(1)
    xs = rng.uniform(-3.0, 3.0, 200_000)
    for x in xs[:50_000]:
        w = oracle.wrap(x)
        assert 0.0 <= w < 1.0
    inside = rng.uniform(0.0, 1.0, 20_000)
    for x in inside:
        assert oracle.wrap(x) == x                              # identity on [0,1)
    for x in xs[:2000]:                                         # exact restatement
        assert oracle.wrap(x) == float(wrap_exact(F(x)))


# ------------------------------------------------------------------------- drift (a2; Eq. 1)
def test_drift_closed_form_constant_velocity():
    s = inputs.make_r1(4096, seed=3)
    n = 10
    out = oracle.drift(s, DT, n)
    exp = np.empty_like(s["pos"])
    for c in range(3):
        for i in range(s["pos"].shape[1]):
            x = F(s["pos"][c, i]) + n * F(DT) * F(s["vel"][c, i])
            exp[c, i] = float(x - math.floor(x))
    assert pdist(out["pos"], exp).max() <= 1e-14                # ~ n * 2^-53
    assert np.array_equal(bits(out["vel"]), bits(s["vel"])) and np.array_equal(out["id"], s["id"])


def test_drift_hand_cases_cross_faces():
    s = r1([[0.999, 0.001, 0.0]], [[2.0, -2.0, -1e-17]])
    one = oracle.drift(s, DT, 1)
    assert one["pos"][0, 0] < 0.002 and abs(one["pos"][0, 0] - 0.001) < 1e-15     # crossed the upper face
    assert one["pos"][1, 0] > 0.998 and abs(one["pos"][1, 0] - 0.999) < 1e-15     # crossed the lower face
    assert one["pos"][2, 0] == 0.0                              # fma gives -1e-20; wrap must give 0.0, not 1.0
    ten = oracle.drift(s, DT, 10)
    assert abs(ten["pos"][0, 0] - 0.019) < 1e-14 and abs(ten["pos"][1, 0] - 0.981) < 1e-14


def test_drift_bit_exact_vs_exact_rational():
    s = inputs.make_r1(48, seed=11)
    s["vel"] *= np.float32(300.0)                               # many face crossings in 3 steps
    out = oracle.drift(s, DT, 3)
    for c in range(3):
        for i in range(48):
            p, v = F(s["pos"][c, i]), F(s["vel"][c, i])
            for _ in range(3):
                p = wrap_exact(rn64(F(DT) * v + p))             # ONE rounding: a true fma
            assert bits(out["pos"][c, i:i + 1])[0] == bits(np.array([to_f64(p)]))[0]


def test_drift_wide_record_double_velocity():
    s = inputs.make_r2(32, seed=5)
    out = oracle.drift(s, DT, 2)
    for c in range(3):
        for i in range(32):
            p, v = F(s["pos"][c, i]), F(s["vel"][c, i])
            for _ in range(2):
                p = wrap_exact(rn64(F(DT) * v + p))
            assert out["pos"][c, i] == float(p)
    for k in ("id", "vel", "acc", "mass", "charge", "flags"):
        assert np.array_equal(bits(out[k]), bits(s[k]))


# ------------------------------------------------------------- symplectic Euler (a4; Q2, Q4; config 2)
def _nonwrapping(n, seed, vmax=0.1):
    rng = np.random.default_rng(seed)
    return r1(rng.uniform(0.3, 0.7, (n, 3)), rng.uniform(-vmax, vmax, (n, 3)).astype(np.float32))


@pytest.mark.parametrize("k", [1.0, 2.5])
def test_symplectic_euler_linear_closed_form(k):
    s = _nonwrapping(256, 2)
    n = 100
    out = oracle.symplectic_euler(s, DT, n, k=k)
    M = np.array([[1.0 - DT * DT * k, DT], [-DT * k, 1.0]])   # kick (new v) then drift with the NEW v
    Mn = np.linalg.matrix_power(M, n)
    x0, v0 = s["pos"] - 0.5, s["vel"].astype(np.float64)
    xe, ve = Mn[0, 0] * x0 + Mn[0, 1] * v0, Mn[1, 0] * x0 + Mn[1, 1] * v0
    assert np.abs(out["pos"] - 0.5 - xe).max() < 2e-7           # float-v rounding dominates
    assert np.abs(out["vel"] - ve).max() < 5e-6
    # the other order (drift, then kick) differs by O(dt): make sure the tolerance separates them
    Mw = np.linalg.matrix_power(np.array([[1.0, DT], [-DT * k, 1.0 - DT * DT * k]]), n)
    assert np.abs(Mw[0, 0] * x0 + Mw[0, 1] * v0 - xe).max() > 1e-5


def test_symplectic_euler_discrete_invariant():
    s = _nonwrapping(512, 4, vmax=0.2)
    out = oracle.symplectic_euler(s, DT, 1000)

    def inv(t):
        x, v = t["pos"] - 0.5, t["vel"].astype(np.float64)
        return x * x + v * v - DT * x * v                       # exact invariant of the kick-drift map

    i0, i1 = inv(s), inv(out)
    # float-v rounding random-walks the invariant by ~sqrt(1000) * 2^-24 * |v|^2 ~ 1e-7..5e-7 (SURVEY 8(c):
    # "with float v it holds to ~1e-6 relative"); dropping the -dt*x*v term would move it by ~4e-5.
    assert np.abs(i1 - i0).max() < 1e-6
    assert np.abs((i1 - i0) + DT * (out["pos"] - 0.5) * out["vel"]).max() > 5e-6   # the cross term matters


def test_symplectic_euler_bit_exact_vs_exact_rational():
    s = inputs.make_r1(40, seed=21)
    s["vel"] *= np.float32(200.0)
    k, ctr, nsteps = 1.0, 0.5, 3
    out = oracle.symplectic_euler(s, DT, nsteps, k=k, center=ctr)
    dtf = rn32(F(DT))
    for c in range(3):
        for i in range(40):
            p, v = F(s["pos"][c, i]), F(s["vel"][c, i])
            for _ in range(nsteps):
                force = rn32(-rn64(F(k) * rn64(p - F(ctr))))    # double subtract, *k, negate, RN to float
                v = rn32(dtf * force + v)                       # float fma, dt_f = (float)dt
                p = wrap_exact(rn64(F(DT) * v + p))             # double fma with the NEW velocity
            assert out["pos"][c, i] == float(p), (c, i)
            assert bits(out["vel"][c, i:i + 1])[0] == bits(np.array([to_f32(v)]))[0], (c, i)


def test_config2_energy_statistics_and_boundedness():
    n = 1 << 16
    s = inputs.make_r1(n, seed=0)
    e0 = oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC)
    assert abs(e0 / n - 1.625) < 0.02                           # KE 1.5 (N(0,1)^3) + PE 3*(1/2)(1/12)
    out = oracle.symplectic_euler(s, DT, 100)
    e1 = oracle.energy(out, oracle.KINETIC_PLUS_HARMONIC)
    assert abs(e1 - e0) / e0 < 1e-3                             # symplectic Euler keeps energy bounded
    assert (out["pos"] >= 0).all() and (out["pos"] < 1).all()
    wrapped = np.abs(out["pos"] - s["pos"]) > 0.5
    assert 0.02 < wrapped.mean() < 0.2                          # the wrap branch is exercised (~7.7 %)
    assert np.array_equal(out["id"], s["id"])


# --------------------------------------------------------------------- RK2 midpoint, masked (a9; Q6-Q8)
def _r2_nonwrapping(n, seed):
    s = inputs.make_r2(n, seed)
    rng = np.random.default_rng(seed)
    s["pos"][:] = rng.uniform(0.35, 0.65, (3, n))
    s["vel"][:] = rng.uniform(-0.1, 0.1, (3, n))
    return s


def test_rk2_linear_closed_form_and_mask():
    s = _r2_nonwrapping(300, 6)
    n, k = 20, 1.75
    out = oracle.rk2_midpoint_masked(s, DT, n, k=k, mask=1)
    active = (s["flags"][0] & 1) != 0
    assert 50 < active.sum() < 250
    w = k / s["mass"][0].astype(np.float64)
    x0, v0 = s["pos"] - 0.5, s["vel"]
    for i in np.nonzero(active)[0]:
        a = 1.0 - DT * DT * w[i] / 2.0
        Mn = np.linalg.matrix_power(np.array([[a, DT], [-DT * w[i], a]]), n)
        xe, ve = Mn[0, 0] * x0[:, i] + Mn[0, 1] * v0[:, i], Mn[1, 0] * x0[:, i] + Mn[1, 1] * v0[:, i]
        assert np.abs(out["pos"][:, i] - 0.5 - xe).max() < 1e-13
        assert np.abs(out["vel"][:, i] - ve).max() < 1e-13
        # acc = midpoint acceleration of the LAST step (Q7): a2 = -w (x_prev + dt/2 v_prev)
        Mp = np.linalg.matrix_power(np.array([[a, DT], [-DT * w[i], a]]), n - 1)
        xp, vp = Mp[0, 0] * x0[:, i] + Mp[0, 1] * v0[:, i], Mp[1, 0] * x0[:, i] + Mp[1, 1] * v0[:, i]
        assert np.abs(out["acc"][:, i] + w[i] * (xp + 0.5 * DT * vp)).max() < 1e-12
    for name in s:                                              # inactive rows and untouched fields: bitwise
        same = bits(out[name]) == bits(s[name])
        assert same[:, ~active].all(), name
        if name in ("id", "mass", "charge", "flags"):
            assert same.all(), name
    assert (out["acc"][:, ~active] == 0).all()


@pytest.mark.parametrize("w", [0.5, 1.0, 2.0])
def test_rk2_exact_energy_growth_factor(w):
    # one-step map is linear; E = v^2/2 + w x^2/2 grows by exactly (1 + dt^4 w^2 / 4) per step
    s = _r2_nonwrapping(64, 8)
    s["flags"][:] = 1
    s["mass"][:] = np.float32(1.0 / w)                          # k = 1 -> w exactly
    n = 20
    out = oracle.rk2_midpoint_masked(s, DT, n, k=1.0)
    e0 = 0.5 * (s["vel"] ** 2 + w * (s["pos"] - 0.5) ** 2).sum(axis=0)
    e1 = 0.5 * (out["vel"] ** 2 + w * (out["pos"] - 0.5) ** 2).sum(axis=0)
    pred = (1.0 + DT ** 4 * w * w / 4.0) ** n - 1.0
    # rounding floor of 20 double steps + the e1/e0 evaluation is a few 2^-52; pred is 1.2e-12 .. 2e-11
    assert np.abs((e1 / e0 - 1.0) - pred).max() < 1.5e-14


def test_rk2_bit_exact_vs_exact_rational_with_wraps():
    s = inputs.make_r2(40, seed=9)
    s["vel"] *= 400.0
    k, ctr, mask, nsteps = 1.0, 0.5, 1, 2
    out = oracle.rk2_midpoint_masked(s, DT, nsteps, k=k, center=ctr, mask=mask)
    hh = F(0.5 * DT)
    for i in range(40):
        if not (int(s["flags"][0, i]) & mask):
            continue
        w = rn64(F(k) / F(s["mass"][0, i]))
        p = [F(s["pos"][c, i]) for c in range(3)]
        v = [F(s["vel"][c, i]) for c in range(3)]
        a2 = [Fraction(0)] * 3
        for _ in range(nsteps):
            a1 = [-rn64(w * rn64(p[c] - F(ctr))) for c in range(3)]
            ph = [wrap_exact(rn64(hh * v[c] + p[c])) for c in range(3)]
            vh = [rn64(hh * a1[c] + v[c]) for c in range(3)]
            a2 = [-rn64(w * rn64(ph[c] - F(ctr))) for c in range(3)]
            p = [wrap_exact(rn64(F(DT) * vh[c] + p[c])) for c in range(3)]
            v = [rn64(F(DT) * a2[c] + v[c]) for c in range(3)]
        for c in range(3):
            assert out["pos"][c, i] == float(p[c]) and out["vel"][c, i] == float(v[c]) and out["acc"][c, i] == float(a2[c])


def test_mass_clamp_is_live():
    u = np.array([0.0, 0.5, 1.0 - 2.0 ** -53, 1.0 - 2.0 ** -30])
    m = inputs.mass_from_uniform(u)
    assert m.dtype == np.float32 and (m < np.float32(2.0)).all() and m[0] == np.float32(0.5)
    assert m[2] == np.nextafter(np.float32(2.0), np.float32(0.0))


# ------------------------------------------------------------------------------------------ energy (a8)
def _load_energy_fixture(golden_dir):
    rows, exp = [], {}
    for line in open(os.path.join(golden_dir, "energy_4particles.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        t = line.split()
        if t[0].startswith("expect_"):
            exp[t[0]] = float(t[1])
        else:
            rows.append([float(x) for x in t])
    a = np.array(rows)
    return r1(a[:, 3:6], a[:, 0:3]), exp


def test_energy_hand_fixture(golden_dir):
    s, exp = _load_energy_fixture(golden_dir)
    assert oracle.energy(s, oracle.KINETIC) == exp["expect_kinetic"] == 18.5
    assert oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC) == exp["expect_total"] == 18.8125
    for order in ([3, 2, 1, 0], [2, 0, 3, 1]):                   # dyadic: exact in any order
        assert oracle.energy(inputs.take(s, np.array(order)), oracle.KINETIC_PLUS_HARMONIC) == 18.8125
    # general k multiplies only the potential part
    assert oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC, k=4.0) == 18.5 + 4.0 * 0.3125


def test_energy_terms_and_compensated_sum():
    n = 3000
    s = inputs.make_r1(n, seed=13)
    k, ctr = 1.0, 0.5
    terms = []
    for i in range(n):
        v = [F(s["vel"][c, i]) for c in range(3)]
        q = rn64(v[0] * v[0])
        q = rn64(v[1] * v[1] + q)
        q = rn64(v[2] * v[2] + q)
        for c in range(3):
            d = rn64(F(s["pos"][c, i]) - F(ctr))
            q = rn64(rn64(F(k) * d) * d + q)
        terms.append(q / 2)
    # per-particle term, bit exact (single-particle calls)
    for i in range(0, n, 97):
        assert oracle.energy(inputs.take(s, np.array([i])), oracle.KINETIC_PLUS_HARMONIC) == float(terms[i])
    exact = sum(terms, Fraction(0))
    got = oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC)
    assert abs(F(got) - exact) <= Fraction(math.ulp(got))       # Neumaier: within one ulp of the exact sum


def test_energy_compensated_sum_large_n_vs_fsum():
    n = 1 << 18
    s = inputs.make_r1(n, seed=0)
    v = s["vel"].astype(np.float64)
    ke_terms = 0.5 * (v ** 2).sum(axis=0)                       # not bit-identical per term (no fma): 1e-15 rel
    got = oracle.energy(s, oracle.KINETIC)
    assert abs(got - math.fsum(ke_terms)) / got < 1e-14
    assert abs(got / n - 1.5) < 0.01



def _r2(pos, vel, acc=None, mass=None, charge=None, flags=None, ids=None):
    pos = np.asarray(pos, np.float64).reshape(-1, 3)
    vel = np.asarray(vel, np.float64).reshape(-1, 3)
    n = pos.shape[0]
    acc = np.zeros((n, 3)) if acc is None else np.asarray(acc, np.float64).reshape(-1, 3)
    return {"id": (np.arange(n, dtype=np.int64) if ids is None else np.asarray(ids, np.int64))[None, :].copy(),
            "pos": np.ascontiguousarray(pos.T), "vel": np.ascontiguousarray(vel.T), "acc": np.ascontiguousarray(acc.T),
            "mass": (np.ones(n, np.float32) if mass is None else np.asarray(mass, np.float32))[None, :].copy(),
            "charge": (np.ones(n, np.float32) if charge is None else np.asarray(charge, np.float32))[None, :].copy(),
            "flags": (np.zeros(n, np.uint8) if flags is None else np.asarray(flags, np.uint8))[None, :].copy()}


def test_energy_r2_hand_fixture(golden_dir):
    """The same 4-particle dyadic fixture stored as the wide record R2 (double vel): 18.5 / 18.8125 with '=='.
    acc, mass, charge, flags and id are filled with values that would change the sum if any were read instead of
    vel / pos (a wrong member in soax_oracle_r2_energy fails here)."""
    s1, exp = _load_energy_fixture(golden_dir)
    s = _r2(s1["pos"].T, s1["vel"].T.astype(np.float64), acc=[[7, 7, 7]] * 4, mass=[3, 5, 9, 17], charge=[-1, 1, -1, 1],
            flags=[1, 2, 3, 4], ids=[100, 200, 300, 400])
    assert oracle.energy(s, oracle.KINETIC) == exp["expect_kinetic"] == 18.5
    assert oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC) == exp["expect_total"] == 18.8125
    for order in ([3, 2, 1, 0], [2, 0, 3, 1]):
        assert oracle.energy(inputs.take(s, np.array(order)), oracle.KINETIC_PLUS_HARMONIC) == 18.8125
    assert oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC, k=4.0) == 18.5 + 4.0 * 0.3125
    assert oracle.energy(s, oracle.KINETIC_PLUS_HARMONIC, k=1.0, center=0.0) == 18.5 + 0.5 * (0.75 + 0.5 + 0.875 + 0.5)
    # component order matters in the fma chain only through rounding; a dropped component changes the value:
    t = _r2([[0.5, 0.5, 0.5]], [[1.0, 2.0, 4.0]])
    assert oracle.energy(t, oracle.KINETIC) == 10.5
    assert oracle.energy(_r2([[0.25, 0.5, 1.0]], [[0, 0, 0]]), oracle.KINETIC_PLUS_HARMONIC) == 0.5 * (0.0625 + 0.25)


def test_energy_r2_terms_and_compensated_sum():
    """Per-particle term of the double-velocity record restated with exact rationals and one rounding per IEEE
    operation (bit for bit), general k and centre; the Neumaier sum within one ulp of the exact sum."""
    n = 2000
    s = inputs.make_r2(n, seed=21)
    s["acc"][:] = np.random.default_rng(3).normal(size=(3, n))         # must not enter the sum
    for kind, k, ctr in ((oracle.KINETIC, 1.0, 0.5), (oracle.KINETIC_PLUS_HARMONIC, 1.0, 0.5), (oracle.KINETIC_PLUS_HARMONIC, 2.5, 0.25)):
        terms = []
        for i in range(n):
            v = [F(s["vel"][c, i]) for c in range(3)]
            q = rn64(v[0] * v[0])
            q = rn64(v[1] * v[1] + q)
            q = rn64(v[2] * v[2] + q)
            if kind == oracle.KINETIC_PLUS_HARMONIC:
                for c in range(3):
                    d = rn64(F(s["pos"][c, i]) - F(ctr))
                    q = rn64(rn64(F(k) * d) * d + q)
            terms.append(q / 2)
        for i in range(0, n, 89):
            assert oracle.energy(inputs.take(s, np.array([i])), kind, k, ctr) == float(terms[i])
        exact = sum(terms, Fraction(0))
        got = oracle.energy(s, kind, k, ctr)
        assert abs(F(got) - exact) <= Fraction(math.ulp(got))
    # double velocities are NOT rounded through float: a value with more than 24 significant bits keeps them
    t = _r2([[0.5, 0.5, 0.5]], [[1.0 + 2.0 ** -40, 0.0, 0.0]])
    assert oracle.energy(t, oracle.KINETIC) == float(rn64(F(1.0 + 2.0 ** -40) ** 2) / 2) != 0.5


# ------------------------------------------------------------------------------ AoS <-> SoA (a6, a7; Q1)
def test_r1_packed_layout_offsets():
    off = np.zeros(7, np.int64)
    oracle.lib().soax_oracle_r1_offsets(off.ctypes.data)
    assert off.tolist() == [0, 4, 12, 20, 28, 32, 36]           # declaration order, no padding (Q1)
    assert oracle.lib().soax_oracle_r1_stride() == 40 == oracle.R1_DTYPE.itemsize
    assert oracle.lib().soax_oracle_r2_stride() == 96 == oracle.R2_DTYPE.itemsize


def test_aos_soa_roundtrip_random_bytes():
    rng = np.random.default_rng(5)
    n = 1001
    raw = rng.integers(0, 256, 40 * n, dtype=np.uint8)          # every bit pattern incl. NaN payloads
    soa = oracle.r1_aos_to_soa(raw)
    rec = raw.view(oracle.R1_DTYPE)                             # numpy's own view of the packed record
    assert np.array_equal(soa["id"][0], rec["id"])
    for c in range(3):
        assert np.array_equal(bits(soa["pos"][c]), bits(np.ascontiguousarray(rec["pos"][:, c])))
        assert np.array_equal(bits(soa["vel"][c]), bits(np.ascontiguousarray(rec["vel"][:, c])))
    assert np.array_equal(oracle.r1_soa_to_aos(soa), raw)       # byte-exact round trip (no padding bytes)


# ------------------------------------------------------- binning (a10..a13; config 5; Q11, Q12, Q16)
def _load_binning_fixture(golden_dir):
    pos, cells, exp = [], [], {}
    for line in open(os.path.join(golden_dir, "binning_6particles.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        t = line.split()
        if t[0] in ("counts", "offsets", "perm", "dest"):
            exp[t[0]] = np.array([int(x) for x in t[1:]], np.uint32)
        else:
            pos.append([float(x) for x in t[:3]])
            cells.append(int(t[3]))
    return np.array(pos), np.array(cells, np.uint32), exp


def test_binning_hand_fixture(golden_dir):
    pos, cells, exp = _load_binning_fixture(golden_dir)
    s = r1(pos, np.zeros_like(pos))
    b = oracle.bin_r1(s, 2)
    assert np.array_equal(b["cell"], cells)
    for key in ("counts", "offsets", "perm", "dest"):
        assert np.array_equal(b[key], exp[key]), key


def _brute_dest(cell):
    n = len(cell)
    return np.array([sum(1 for j in range(n) if cell[j] < cell[i]) + sum(1 for j in range(i) if cell[j] == cell[i])
                     for i in range(n)], np.uint32)


def _positions_for_cells(cells, G, rng):
    cells = np.asarray(cells)
    idx = np.stack([cells // (G * G), (cells // G) % G, cells % G], axis=1)
    return (idx + rng.uniform(0.0, 1.0, idx.shape)) / G


@pytest.mark.parametrize("case", ["random", "one_cell", "sorted", "reversed", "n1", "n63", "two_cells"])
def test_binning_brute_force_small(case):
    rng = np.random.default_rng(17)
    G = 4
    if case == "random":
        pos = rng.uniform(0, 1, (64, 3))
    elif case == "one_cell":
        pos = _positions_for_cells([37] * 50, G, rng)
    elif case == "sorted":
        pos = _positions_for_cells(np.sort(rng.integers(0, 64, 61)), G, rng)
    elif case == "reversed":
        pos = _positions_for_cells(np.sort(rng.integers(0, 64, 62))[::-1], G, rng)
    elif case == "n1":
        pos = np.array([[0.99, 0.0, 0.5]])
    elif case == "n63":
        pos = rng.uniform(0, 1, (63, 3))
    else:
        pos = _positions_for_cells(rng.choice([5, 60], 57), G, rng)
    n = pos.shape[0]
    s = r1(pos, rng.normal(size=(n, 3)), ids=rng.permutation(n))
    b = oracle.bin_r1(s, G)
    i = np.minimum((pos * G).astype(np.int64), G - 1)
    cell = (i[:, 0] * G + i[:, 1]) * G + i[:, 2]                 # x slowest, z fastest (Q11)
    assert np.array_equal(b["cell"], cell)
    assert np.array_equal(b["counts"], np.bincount(cell, minlength=G ** 3))
    dest = _brute_dest(cell)                                     # the O(N^2) definition
    assert np.array_equal(b["dest"], dest)
    perm = np.empty(n, np.uint32)
    perm[dest] = np.arange(n)
    assert np.array_equal(b["perm"], perm)
    new = oracle.permute_r1(s, b["perm"])
    for name in s:
        assert np.array_equal(bits(new[name]), bits(s[name][:, b["perm"]])), name


def test_binning_invariants_and_stable_argsort_large():
    n = 200_003
    s = inputs.make_r1(n, seed=7)
    s = oracle.drift(s, DT, 1)
    G = 64
    b = oracle.bin_r1(s, G)
    assert int(b["counts"].sum()) == n
    assert b["offsets"][0] == 0 and np.array_equal(np.diff(b["offsets"]), b["counts"][:-1])
    assert int(b["offsets"][-1]) + int(b["counts"][-1]) == n
    assert np.array_equal(b["perm"], np.argsort(b["cell"], kind="stable").astype(np.uint32))
    assert np.array_equal(np.sort(b["perm"]), np.arange(n, dtype=np.uint32))
    sc = b["cell"][b["perm"]]
    assert (np.diff(sc.astype(np.int64)) >= 0).all()
    same = np.diff(sc.astype(np.int64)) == 0
    assert (np.diff(b["perm"].astype(np.int64))[same] > 0).all()  # ascending source index within a cell
    assert np.array_equal(b["dest"][b["perm"]], np.arange(n, dtype=np.uint32))
    new = oracle.permute_r1(s, b["perm"])
    assert np.array_equal(np.sort(new["id"][0]), np.arange(n, dtype=np.int32))   # ids stay a permutation
    assert np.array_equal(new["id"][0], s["id"][0][b["perm"]])


def test_cell_index_extremes():
    top = 1.0 - 2.0 ** -53
    s = r1([[top, top, top], [0.0, 0.0, 0.0], [0.5, 0.25, 0.125]], np.zeros((3, 3)))
    b = oracle.bin_r1(s, 64, want_perm=False)
    assert b["cell"].tolist() == [64 ** 3 - 1, 0, (32 * 64 + 16) * 64 + 8]       # Q16: largest double < 1 -> 63


# -------------------------------------------------------------- paper-replica benchmark
@pytest.mark.parametrize("size_extra", [0, 32])
def test_b6_euler_bit_exact(size_extra):
    s = inputs.make_b6(50, seed=4)
    dt = np.float32(1e-3)
    p1, v1 = oracle.b6_euler(s["pos"], s["vel"], size_extra, float(dt), 3)
    assert np.array_equal(bits(v1), bits(s["vel"]))
    for c in range(3):
        for i in range(50):
            x, v = F(s["pos"][c, i]), F(s["vel"][c, i])
            for _ in range(3):
                x = rn32(F(dt) * v + x)
            assert bits(p1[c, i:i + 1])[0] == bits(np.array([to_f32(x)]))[0]


# ------------------------------------------------------------------------------- generators (sanity only)
def test_generators_sanity():
    n = 1 << 16
    s = inputs.make_r1(n, seed=0)
    assert np.array_equal(np.sort(s["id"][0]), np.arange(n, dtype=np.int32))
    assert (s["pos"] >= 0).all() and (s["pos"] < 1).all() and abs(s["pos"].mean() - 0.5) < 0.01
    assert abs(s["vel"].mean()) < 0.02 and abs(s["vel"].std() - 1.0) < 0.02
    t = inputs.make_r1(n // 2, seed=0)
    assert np.array_equal(t["pos"], s["pos"][:, :n // 2])        # a prefix of a larger set is the smaller set
    assert not np.array_equal(inputs.make_r1(n, seed=7)["pos"], s["pos"])
    for m in (1, 2, 3, 1000, 65537):
        p = inputs.random_permutation(5, m, np.int64)
        assert np.array_equal(np.sort(p), np.arange(m))
    r2 = inputs.make_r2(n, seed=0)
    assert set(np.unique(r2["charge"])) == {-1.0, 1.0} and (r2["acc"] == 0).all()
    assert r2["mass"].min() >= 0.5 and r2["mass"].max() < 2.0
    assert 0.45 < (r2["flags"][0] & 1).mean() < 0.55
    assert [inputs.shard_range(10, r, 3) for r in range(3)] == [(0, 4), (4, 7), (7, 10)]
