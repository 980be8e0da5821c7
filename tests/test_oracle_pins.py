"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test names the passage it checks.  A plausible mistake in oracle/mmc_oracle.c (dropped term,
wrong sign/index, transposed operand) is meant to fail at least one of these.
"""
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
KB, MUB = O.KB, O.MUB


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------------------ O2 Philox
def test_philox_known_answers():
    for r in _rows("philox_kat.txt"):
        v = [int(x, 16) for x in r]
        assert O.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_uniform_mapping_is_fp32_exact_and_open():
    for x in (0, 1, 511, 512, 0xFFFFFFFF, 0x80000000, 0x12345678):
        u = O.u01(x)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u                      # exactly representable in fp32
    assert O.u01(0) == 2.0 ** -24 and O.u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    u = O.cell_uniforms(0x5EED0001, 7, 5)                      # 0.98704737, 0.01140862, ...
    assert np.allclose(u, [0.98704737, 0.01140862, 0.54913157, 0.80376559], atol=1e-8)


# ------------------------------------------------------------------------------ O1 thermal
def test_thermal_probe_values():
    for T, Tc, V, Ms0, q, val, tol in _rows("thermal_probe.txt"):
        th = O.thermal(float(T), float(Tc), MUB, float(V), float(Ms0))
        assert th[q] == pytest.approx(float(val), rel=float(tol)), (T, Tc, q)


def test_me_against_mpmath_root():
    """Eq. (9) with H_ext = 0 solved independently by mpmath.findroot at 40 digits."""
    mp.mp.dps = 40
    for T, Tc in ((300, 870), (500, 870), (679, 680), (650, 700), (10, 700), (699.9, 700)):
        a = mp.mpf(3) * Tc / T
        x0 = float(np.sqrt(max(1e-6, 5.0 / 3.0 * (1 - T / Tc)))) if T > 0.5 * Tc else 0.95
        root = mp.findroot(lambda m: mp.coth(a * m) - 1 / (a * m) - m, x0)
        assert O.me_of_T(T, Tc) == pytest.approx(float(root), rel=1e-12)
    assert O.me_of_T(700, 700) == 0.0 and O.me_of_T(800, 700) == 0.0


def test_langevin_and_derivative_against_mpmath():
    mp.mp.dps = 40
    for x in (1e-6, 1e-4, 5e-3, 0.0999, 0.1001, 0.3, 3.0, 30.0, 400.0):
        B = mp.coth(x) - 1 / mp.mpf(x)
        Bp = 1 / mp.mpf(x) ** 2 - 1 / mp.sinh(x) ** 2
        assert O.langevin(x) == pytest.approx(float(B), rel=2e-10)
        assert O.langevin_prime(x) == pytest.approx(float(Bp), rel=2e-9)


def test_chi_curie_weiss_and_series_near_Tc():
    """Above Tc Eq. (8) is mu/(3 kB (T - Tc)); just below, mu/(6 kB (Tc - T)) and me^2 = (5/3)(Tc-T)/Tc to
    leading order; both branches of Eq. (7) meet at c2 = 0, c4 = (9/20) V Ms0/mu."""
    Tc, V, Ms0 = 680.0, 1.25e-25, 8e5
    for T in (681.0, 700.0, 1000.0):
        th = O.thermal(T, Tc, MUB, V, Ms0)
        assert th["chi"] == pytest.approx(MUB / (3 * KB * (T - Tc)), rel=1e-12)
        assert th["c2"] == pytest.approx(V * Ms0 * 3 * KB * (T - Tc) / (2 * MUB * KB * T), rel=1e-12)
    for d in (0.1, 0.01):
        th = O.thermal(Tc - d, Tc, MUB, V, Ms0)
        assert th["chi"] == pytest.approx(MUB / (6 * KB * d), rel=5 * d / Tc + 1e-3)
        assert th["me"] ** 2 == pytest.approx(5.0 / 3.0 * d / Tc, rel=5 * d / Tc + 1e-3)
    lim = 9.0 / 20.0 * V * Ms0 / MUB
    at = O.thermal(Tc, Tc, MUB, V, Ms0)
    assert at["c2"] == 0.0 and at["c4"] == pytest.approx(lim, rel=1e-14)
    for d in (-1e-3, 1e-3):
        th = O.thermal(Tc + d, Tc, MUB, V, Ms0)
        assert th["c4"] == pytest.approx(lim, rel=1e-4) and abs(th["c2"]) < 0.05
    with pytest.raises(ValueError):
        O.thermal(0.0, Tc, MUB, V, Ms0)


def test_longitudinal_quartic_is_exponent_of_eq7():
    """c4 m^4 + c2 m^2 + c0 must equal the two exponents of Eq. (7) written out literally."""
    V, Ms0 = 1.25e-25, 8e5
    for T, Tc in ((300.0, 870.0), (679.0, 680.0)):
        th = O.thermal(T, Tc, MUB, V, Ms0)
        for m in (0.05, 0.5, 0.9):
            lit = V * Ms0 / (8 * th["chi"] * th["me"] ** 2 * KB * T) * (m * m - th["me"] ** 2) ** 2
            assert th["c4"] * m ** 4 + th["c2"] * m ** 2 + th["c0"] == pytest.approx(lit, rel=1e-9, abs=1e-9)
    T, Tc = 700.0, 680.0
    th = O.thermal(T, Tc, MUB, V, Ms0)
    for m in (0.01, 0.1):
        lit = V * Ms0 * m * m / (2 * th["chi"] * KB * T) * (1 + 3 * Tc * m * m / (10 * (T - Tc)))
        assert th["c4"] * m ** 4 + th["c2"] * m ** 2 == pytest.approx(lit, rel=1e-12)


def test_sigma_eq13_and_cap():
    V, Ms0, Tc = 8e-27, 6e5, 700.0
    th = O.thermal(200.0, Tc, MUB, V, Ms0)
    assert th["sigma13"] == pytest.approx(2 * th["me"] * np.sqrt(th["chi"] * KB * 200.0 / (V * Ms0)), rel=1e-13)
    assert O.thermal(650.0, Tc, MUB, V, Ms0)["sigma13"] == 0.03       # cap
    assert O.thermal(750.0, Tc, MUB, V, Ms0)["sigma13"] == 0.03       # constant above Tc


# ------------------------------------------------------------------------------ O3 trial move
def test_trial_move_geometry():
    rng = np.random.default_rng(1)
    for _ in range(300):
        m = rng.normal(size=3) * rng.uniform(0.01, 1.0)
        if rng.uniform() < 0.3:
            m[rng.integers(3)] = 0.0                                   # exercise the axis choice / ties
        u = rng.uniform(size=3)
        cone = np.deg2rad(rng.uniform(0.5, 180.0)); w = 1 - np.cos(cone)
        sig = rng.uniform(0, 0.05)
        dm, f = O.trial(m, u, w, sig)
        mp_ = m + dm
        L, Lp = np.linalg.norm(m), np.linalg.norm(mp_)
        assert f == pytest.approx(1 + sig * (2 * u[2] - 1), rel=1e-15)
        assert Lp / L == pytest.approx(f, rel=1e-13)                   # |m'|/|m| = f exactly
        cos_t = np.dot(m, mp_) / (L * Lp)
        assert cos_t == pytest.approx(1 - u[0] * w, abs=1e-13)         # polar angle from u_cos only
        assert cos_t >= np.cos(cone) - 1e-13                           # inside the cone (PAPER.md:92 step 1)
    dm, f = O.trial([0.3, -0.2, 0.5], [0.3, 0.7, 0.123], 0.2, 0.0)     # sigma = 0 conserves |m|
    assert f == 1.0 and np.linalg.norm(np.array([0.3, -0.2, 0.5]) + dm) == pytest.approx(np.linalg.norm([0.3, -0.2, 0.5]), rel=1e-14)


def test_trial_move_uniform_on_cap_and_azimuth():
    """Reading G6: uniform in solid angle on the cap => cos(theta) uniform on [cos(theta_c), 1] and the
    azimuth uniform; the azimuth must advance with u_phi in a right-handed frame (t1, t2, n)."""
    m = np.array([0.2, 0.5, -0.4]); n = m / np.linalg.norm(m)
    w = 1 - np.cos(np.deg2rad(40.0))
    a = int(np.argmin(np.abs(m))); e = np.eye(3)[a]
    t1 = np.cross(e, n); t1 /= np.linalg.norm(t1); t2 = np.cross(n, t1)
    for uphi in (0.0, 0.125, 0.25, 0.5, 0.8):
        dm, _ = O.trial(m, [0.6, uphi, 0.5], w, 0.0)
        d = (m + dm) / np.linalg.norm(m + dm)
        az = np.arctan2(np.dot(d, t2), np.dot(d, t1)) % (2 * np.pi)
        assert az == pytest.approx((2 * np.pi * uphi) % (2 * np.pi), abs=1e-12)


# ------------------------------------------------------------------------------ helpers for meshes
def _mesh(nx, ny, nz, pbc, mats, reg=None, T=300.0, Tcell=None, inter=1, d=(5e-9, 5e-9, 5e-9), seed=3, B=(0, 0, 0),
          cone=30.0, sigma=-1.0, store_fp32=False):
    s = O.OracleMMC(nx, ny, nz, *d, pbc_mask=pbc, store_fp32=store_fp32)
    s.set_material(mats, reg); s.set_exchange_coupling(inter); s.set_temperature(T, Tcell)
    s.set_field(*B); s.set_move(cone, sigma, False); s.set_seed(seed)
    return s


def _rand_m(rng, N, lo=0.3, hi=1.0):
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    return (v * rng.uniform(lo, hi, N)).astype(np.float32)


# ------------------------------------------------------------------------------ O4 / O8 energies
@pytest.mark.parametrize("shape,pbc", [((4, 4, 1), 0b011), ((4, 2, 2), 0b111), ((3, 4, 2), 0b010), ((5, 3, 1), 0), ((2, 2, 1), 0)])
def test_local_dF_equals_global_dE_bruteforce(shape, pbc):
    """O4 vs O8 (PAPER.md:76-79 factor 2; Eq. (11), (15), (7)): for every cell and random trial vectors the
    local dF (all terms but demag) equals E_total(after) - E_total(before) recomputed from scratch."""
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(11 + N + pbc)
    mats = [O.Material(), O.Material(Ms0=8e5, A0=1.3e-11, K1=5e5, ax=0.3, ay=-0.2, az=0.9, D0=2.5e-3, Tc=870.0),
            O.Material(Ms0=6e5, A0=1.3e-11, K1=-2e5, ax=1.0, ay=0.0, az=0.0, D0=2.5e-3, Tc=500.0,
                       K1c=4.8e4, K2c=-1e4, c1x=1.0, c1y=0.4, c1z=-0.2, c2x=0.1, c2y=1.0, c2z=0.3)]    # + cubic, Eq. (12)
    reg = rng.integers(0, 3, N).astype(np.int32); reg[0] = 1
    Tcell = rng.uniform(250, 650, N).astype(np.float32)
    for inter in (1, 0):
        s = _mesh(nx, ny, nz, pbc, mats, reg, Tcell=Tcell, inter=inter, d=(5e-9, 4e-9, 3e-9), B=(0.1, -0.2, 0.3))
        m0 = _rand_m(rng, N); s.set_m(*m0)
        for c in range(N):
            if reg[c] == 0:
                continue
            i, j, k = c % nx, (c // nx) % ny, c // (nx * ny)
            dm = rng.normal(size=3) * 0.3
            ob = s.observables()
            t = s.cell_dF(i, j, k, dm)
            Eb = sum(ob[q] for q in ("E_ex", "E_an", "E_zee", "E_dmi", "E_long"))
            for a in range(3):
                s.m[a][c] += dm[a]
            oa = s.observables()
            Ea = sum(oa[q] for q in ("E_ex", "E_an", "E_zee", "E_dmi", "E_long"))
            for a in range(3):
                s.m[a][c] -= dm[a]
            beta = 1.0 / (KB * float(Tcell[c]))
            for q, name in ((0, "E_ex"), (1, "E_an"), (2, "E_zee"), (3, "E_dmi"), (5, "E_long")):
                scale = max(abs(oa[name]), abs(ob[name]), 1e-30)
                assert t[q] / beta == pytest.approx(oa[name] - ob[name], abs=1e-11 * scale), (name, c, inter)
            assert t[4] == 0.0
            assert (t.sum()) / beta == pytest.approx(Ea - Eb, abs=1e-11 * max(abs(Ea), abs(Eb)))


def test_exchange_is_textbook_heisenberg_on_uniform_state():
    """Uniform m: E_ex = 0, and rotating one cell by angle a costs n_nb * 2 (A0 V/h^2) |m|^2 (1 - cos a)
    (pair energy (A0 V/h^2)|m_i - m_j|^2 per bond; the factor 2 of PAPER.md:79 in the local form)."""
    s = _mesh(4, 4, 1, 0b011, [O.Material(Ms0=8e5, A0=1.3e-11, Tc=870.0)])
    N = 16; m = np.zeros((3, N), dtype=np.float32); m[2] = 0.8; s.set_m(*m)
    assert s.observables()["E_ex"] == 0.0
    a = 0.3; L = float(np.float32(0.8))
    dm = np.array([L * np.sin(a), 0.0, L * (np.cos(a) - 1)])
    t = s.cell_dF(1, 1, 0, dm)
    V, h = 1.25e-25, 5e-9
    expect = 4 * 2 * (1.3e-11 * V / h ** 2) * L * L * (1 - np.cos(a))
    assert t[0] * KB * 300.0 == pytest.approx(expect, rel=1e-12)


def test_zeeman_and_demag_term_signs():
    """dF_zee = -V Ms0 dm.B (lower energy when rotating toward the field); Eq. (14): dF_d = -V mu0 dM.H_d."""
    s = _mesh(2, 2, 1, 0, [O.Material(Ms0=8e5, Tc=870.0)], B=(0, 0, 0.5))
    m = np.zeros((3, 4), dtype=np.float32); m[0] = 0.8; s.set_m(*m)
    t = s.cell_dF(0, 0, 0, np.array([0.0, 0.0, 0.1]))
    assert t[2] == pytest.approx(-(1.25e-25 * 8e5 * 0.1 * 0.5) / (KB * 300.0), rel=1e-13)
    s.demag_enabled = True
    s.bd = [np.full(4, 0.0), np.full(4, 0.02), np.full(4, 0.0)]
    t = s.cell_dF(1, 1, 0, np.array([0.0, -0.1, 0.0]))
    assert t[4] == pytest.approx(+(1.25e-25 * 8e5 * 0.1 * 0.02) / (KB * 300.0), rel=1e-13)


def test_dmi_prefers_the_chirality_eq15_selects():
    """Eq. (15) literal sign (G7): for D0 > 0 a Neel spiral m = (sin qx, 0, cos qx) has E_dmi = -D0 V q |m|^2
    per cell (continuum limit), the opposite spiral +; checks sign, index and 1/(2h) of the central difference."""
    nx, h, D0 = 64, 2e-9, 2.5e-3
    s = _mesh(nx, 2, 1, 0b011, [O.Material(Ms0=6e5, A0=0.0, D0=D0, Tc=700.0)], d=(h, h, h))
    q = 2 * np.pi / (nx * h)
    x = (np.arange(nx) + 0.5) * h
    for sgn in (+1, -1):
        mx = np.tile(np.sin(sgn * q * x), 2); mz = np.tile(np.cos(q * x), 2)
        s.set_m(mx, np.zeros_like(mx), mz)
        E = s.observables()["E_dmi"]
        # m.(z div m - grad mz) = mz dmx/dx - mx dmz/dx = sgn q ; discrete derivative sin(qh)/h
        assert E == pytest.approx(-D0 * h ** 3 * sgn * np.sin(q * h) / h * 2 * nx, rel=1e-6)


# ------------------------------------------------------------------------------ O5 acceptance
def test_acceptance_rule_eq5_and_detailed_balance_ratio():
    """Eq. (5): accept iff u < (mB/mA)^4 exp(-dF).  Eq. (3)+(4): A(A->B)/A(B->A) = (mB/mA)^4 exp(-dF)."""
    rng = np.random.default_rng(5)
    mat = [O.Material(Ms0=8e5, A0=1.3e-11, K1=5e5, D0=1e-3, Tc=870.0)]
    s = _mesh(4, 4, 1, 0b011, mat, T=600.0, B=(0.0, 0.1, 0.2), cone=25.0, sigma=0.04, seed=77)
    m0 = _rand_m(rng, 16, 0.5, 0.8); s.set_m(*m0)
    before = [a.copy() for a in s.m]
    d = s.colour_pass(0, dump=True)
    red = [(c % 4 + c // 4) % 2 == 0 for c in range(16)]
    n_checked = 0
    for c in range(16):
        if not red[c]:
            assert np.isnan(d["margin"][c])
            continue
        u = O.cell_uniforms(77, 0, c)
        mA = np.array([before[a][c] for a in range(3)])
        dm, f = O.trial(mA, u[:3], 2 * np.sin(np.deg2rad(25.0) / 2) ** 2, 0.04)
        assert np.allclose(dm, d["dm"][c], atol=1e-15)
        dF = d["terms"][c].sum()
        ratio = f ** 4 * np.exp(-dF)
        assert bool(d["accepted"][c]) == (u[3] < ratio)
        assert d["margin"][c] == pytest.approx(np.log(u[3]) - np.log(ratio), abs=1e-9)
        # reverse move from B back to A with everything else unchanged
        sB = _mesh(4, 4, 1, 0b011, mat, T=600.0, B=(0.0, 0.1, 0.2), cone=25.0, sigma=0.04)
        mB = [a.copy() for a in before]
        for a in range(3):
            mB[a][c] += dm[a]
        sB.m = mB
        tB = sB.cell_dF(c % 4, c // 4, 0, -dm)
        rB = (1 / f) ** 4 * np.exp(-tB.sum())
        assert min(1, ratio) / min(1, rB) == pytest.approx(ratio, rel=1e-9)
        n_checked += 1
        got = np.array([s.m[a][c] for a in range(3)])
        assert np.allclose(got, mA + dm if d["accepted"][c] else mA, atol=0)
    assert n_checked == 8


def test_checkerboard_order_independence_and_colouring():
    """O6: within a colour no cell reads another cell of that colour, so any visiting order gives
    bit-identical states; every cell gets exactly one trial per sweep."""
    rng = np.random.default_rng(9)
    mat = [O.Material(), O.Material(Ms0=6e5, A0=1e-11, K1=8e5, D0=2.5e-3, Tc=700.0)]
    nx, ny, nz = 6, 4, 2; N = nx * ny * nz
    reg = (rng.uniform(size=N) > 0.15).astype(np.int32)
    m0 = _rand_m(rng, N)
    out = []
    for trial_order in range(3):
        s = _mesh(nx, ny, nz, 0b011, mat, reg, T=500.0, B=(0, 0, 0.1), cone=40.0, seed=5, store_fp32=True)
        s.set_m(*m0)
        for sweep in range(3):
            for col in (0, 1):
                order = None if trial_order == 0 else rng.permutation(N)
                s.colour_pass(col, order=order)
            s.sweep += 1
        assert s.trials == 3 * int(reg.sum())
        out.append(np.stack(s.m))
    assert np.array_equal(out[0], out[1]) and np.array_equal(out[0], out[2])
    assert not np.array_equal(out[0], m0.astype(np.float64))


def test_empty_cells_never_move_and_are_not_counted():
    mat = [O.Material(), O.Material(Ms0=8e5, A0=1.3e-11, Tc=870.0)]
    reg = np.array([1, 0, 1, 1, 0, 1, 1, 1, 0], dtype=np.int32)
    s = _mesh(3, 3, 1, 0, mat, reg, cone=60.0)
    m = np.zeros((3, 9), dtype=np.float32); m[2] = reg * 0.86
    s.set_m(*m); s.run(5)
    assert s.trials == 5 * 6
    assert all(np.all(s.m[a][reg == 0] == 0.0) for a in range(3))


def test_adaptive_cone_controller():
    """PAPER.md:100 + G11: checked every 100 iterations, +-1 degree outside 0.5 +- 0.05."""
    s = _mesh(8, 8, 1, 0b011, [O.Material(Ms0=8e5, A0=1.3e-11, K1=5e5, Tc=870.0)], cone=30.0)
    s.adaptive = True
    rng = np.random.default_rng(2); s.set_m(*(0.8675 * _rand_m(rng, 64, 1.0, 1.0)))
    s.run(99); assert s.cone_deg == 30.0
    rate = s._win_acc / s._win_tri
    s.run(1)
    assert s.cone_deg == (31.0 if rate > 0.55 else 29.0 if rate < 0.45 else 30.0)
    s.run(3900)
    s2 = s.cone_deg
    s.run(2000)   # converged: acceptance near 0.5, cone fluctuates by ~1 deg
    assert 1.0 <= s.cone_deg < 30.0 and abs(s.cone_deg - s2) <= 3.0
    assert 0.40 < s._win_acc / max(1, s._win_tri) < 0.60 or s._win_tri == 0


# ------------------------------------------------------------------------------ equilibrium pins
def _run_independent_cells(T, Tc, B, cone, sigma, n_side, n_sweeps, burn, seed, m_init, every=1):
    """A0 = 0, K1 = 0: n_side^2 independent single-cell chains (single-domain pins of PAPER.md:108-114)."""
    s = _mesh(n_side, n_side, 1, 0, [O.Material(Ms0=8e5, A0=0.0, Tc=Tc)], T=T, B=B, cone=cone, sigma=sigma, seed=seed)
    rng = np.random.default_rng(seed)
    s.set_m(*(m_init * _rand_m(rng, n_side * n_side, 1.0, 1.0)))
    acc_len = []; acc_cos = []; acc_mz = []
    for it in range(n_sweeps):
        s.sweep_once()
        if it >= burn and (it - burn) % every == 0:
            L = np.sqrt(s.m[0] ** 2 + s.m[1] ** 2 + s.m[2] ** 2)
            acc_len.append(L.mean()); acc_cos.append((s.m[2] / L).mean()); acc_mz.append(s.m[2].mean())
    return np.mean(acc_len), np.mean(acc_cos), np.mean(acc_mz), s


def test_single_cell_langevin_angle_distribution():
    """Fixed length (sigma = 0), Zeeman only: <cos theta> = coth(xi) - 1/xi, xi = V Ms0 |m| B / kB T."""
    T, L = 300.0, 0.8675
    B = 3.0 * KB * T / (1.25e-25 * 8e5 * float(np.float32(L)))
    _, c, _, s = _run_independent_cells(T, 870.0, (0, 0, B), 60.0, 0.0, 32, 1500, 300, 21, L)
    assert c == pytest.approx(1 / np.tanh(3.0) - 1 / 3.0, abs=2.5e-3)
    Lf = np.sqrt(s.m[0] ** 2 + s.m[1] ** 2 + s.m[2] ** 2)
    rng = np.random.default_rng(21)                                  # same draw as the initial state
    m0 = (L * _rand_m(rng, 1024, 1.0, 1.0)).astype(np.float32).astype(np.float64)
    assert np.allclose(Lf, np.linalg.norm(m0, axis=0), rtol=1e-12)   # |m| conserved when sigma = 0


def test_single_cell_uniaxial_angle_distribution():
    """Fixed length, uniaxial anisotropy only: <cos^2> = int x^2 e^{k x^2} / int e^{k x^2}, k = V Kq |m|^2/kBT."""
    T, Tc, L = 300.0, 870.0, 0.8675
    me = O.me_of_T(T, Tc); Lf = float(np.float32(L))
    K1 = 2.5 * KB * T / (1.25e-25 * me * Lf * Lf)
    s = _mesh(32, 32, 1, 0, [O.Material(Ms0=8e5, A0=0.0, K1=K1, Tc=Tc)], T=T, cone=60.0, sigma=0.0, seed=8)
    rng = np.random.default_rng(8); s.set_m(*(L * _rand_m(rng, 1024, 1.0, 1.0)))
    acc = []
    for it in range(1500):
        s.sweep_once()
        if it >= 300:
            acc.append(((s.m[2] / Lf) ** 2).mean())
    num = integrate.quad(lambda x: x * x * np.exp(2.5 * x * x), -1, 1)[0]
    den = integrate.quad(lambda x: np.exp(2.5 * x * x), -1, 1)[0]
    assert np.mean(acc) == pytest.approx(num / den, abs=3e-3)


def _eq7_mean(T, Tc, V=1.25e-25, Ms0=8e5):
    th = O.thermal(T, Tc, MUB, V, Ms0)
    if T < Tc:
        w = lambda m: m * m * np.exp(-V * Ms0 / (8 * th["chi"] * th["me"] ** 2 * KB * T) * (m * m - th["me"] ** 2) ** 2)
    else:
        w = lambda m: m * m * np.exp(-V * Ms0 * m * m / (2 * th["chi"] * KB * T) * (1 + 3 * Tc * m * m / (10 * (T - Tc))))
    pts = [0.01, 0.02, 0.05, 0.1, 0.2, 0.5, 0.8, 0.9, 1.0]
    kw = dict(points=pts, limit=400, epsabs=0, epsrel=1e-12)
    return integrate.quad(lambda m: m * w(m), 0, 1.5, **kw)[0] / integrate.quad(w, 0, 1.5, **kw)[0]


def test_eq7_quadrature_matches_golden_means():
    for T, m7, _, _ in _rows("length_means.txt"):
        if float(T) == 680.0:
            continue
        assert _eq7_mean(float(T), 680.0) == pytest.approx(float(m7), rel=2e-5)


@pytest.mark.parametrize("T,idx", [(679.0, 1), (700.0, 3)])
def test_length_distribution_near_and_above_Tc(T, idx):
    """PAPER.md:108 / Eq. (7): the literal (m_B/m_A)^4 chain (reading G1) reproduces the m^2 exp(-F_l/kT) length
    distribution below and above Tc; its exact mean lies ~0.14 sigma (relative) above the Eq. (7) mean."""
    row = _rows("length_means.txt")[idx]
    m7, chain03 = float(row[1]), float(row[2])
    mean_len, _, _, s = _run_independent_cells(T, 680.0, (0, 0, 0), 60.0, 0.03, 64, 9000, 3000, 31, m7, every=10)
    assert mean_len == pytest.approx(chain03, rel=6e-3)
    assert mean_len == pytest.approx(_eq7_mean(T, 680.0), rel=1.2e-2)
    # me itself is NOT the mean: 0.0495 vs 0.1027 at 679 K; 0 vs 0.050 at 700 K
    assert abs(mean_len - O.me_of_T(T, 680.0)) > 0.04
    L = np.sqrt(s.m[0] ** 2 + s.m[1] ** 2 + s.m[2] ** 2)
    assert L.max() < 1.0                                              # P(|M| > Ms0) ~ 0


def test_length_far_below_Tc_tracks_me():
    """300 K, Tc 680: chain, Eq. (7) and me agree to ~2e-5 (SURVEY pin: 0.820897 / 0.820883 / 0.820881)."""
    mean_len, _, _, _ = _run_independent_cells(300.0, 680.0, (0, 0, 0), 30.0, -1.0, 32, 1500, 500, 4, 0.82088)
    assert mean_len == pytest.approx(0.820897, abs=1.5e-4)
    assert mean_len == pytest.approx(_eq7_mean(300.0, 680.0), abs=1.5e-4)


def test_compound_move_joint_length_and_angle():
    """Single cell near Tc in a strong field (T = 679 K, Tc = 680 K, B_z = 1 T): density
    m^2 exp(-(c4 m^4 + c2 m^2)) sin(th) exp(xi0 m cos th); theta integrates to 2 sinh(xi0 m)/(xi0 m)."""
    T, Tc, V, Ms0 = 679.0, 680.0, 1.25e-25, 8e5
    th = O.thermal(T, Tc, MUB, V, Ms0); xi0 = V * Ms0 * 1.0 / (KB * T)
    rho = lambda m: m * m * np.exp(-(th["c4"] * m ** 4 + th["c2"] * m * m)) * 2 * np.sinh(xi0 * m) / (xi0 * m)
    Z = integrate.quad(rho, 1e-9, 1.0)[0]
    lang = lambda x: 1 / np.tanh(x) - 1 / x
    mean_len_q = integrate.quad(lambda m: m * rho(m), 1e-9, 1.0)[0] / Z
    mean_cos_q = integrate.quad(lambda m: lang(xi0 * m) * rho(m), 1e-9, 1.0)[0] / Z
    mean_mz_q = integrate.quad(lambda m: m * lang(xi0 * m) * rho(m), 1e-9, 1.0)[0] / Z
    assert (mean_len_q, mean_cos_q, mean_mz_q) == pytest.approx((0.10666, 0.34384, 0.03978), abs=2e-5)  # SURVEY pin
    ml, mc, mz, _ = _run_independent_cells(T, Tc, (0, 0, 1.0), 60.0, 0.03, 64, 8000, 2500, 13, 0.1, every=10)
    assert ml == pytest.approx(mean_len_q, rel=8e-3)
    assert mc == pytest.approx(mean_cos_q, abs=4e-3)
    assert mz == pytest.approx(mean_mz_q, rel=1.5e-2)


# ------------------------------------------------------------------------------------------------ chunked convergence
def _relax_case(seed=4242):
    import workloads as W
    wl = W.cfg2(nx=12, ny=10)
    wl.demag = False; wl.adaptive_cone = False; wl.seed = seed
    o = O.OracleMMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, store_fp32=True)
    W.configure(o, wl, O.Material)
    return wl, o


def test_relax_driver_follows_the_papers_protocol():
    """The driver of PAPER.md:135 pinned against its own definition written out by hand: chunk averages = plain means of
    the per-iteration cell means of a replayed run; at least two chunks; stops at the first chunk >= 2 whose average
    along the field differs from the previous one by <= threshold; never more than max_chunks."""
    wl, o = _relax_case()
    r = o.relax((1.0, 0.0, 0.0), chunk_sweeps=7, min_chunks=2, max_chunks=6, threshold=1e-4)
    # replay by hand with the same Philox stream
    wl2, o2 = _relax_case()
    per_sweep = []
    for _ in range(r["sweeps"]):
        o2.run(1)
        per_sweep.append(o2.m[0].mean())
    chunks = np.array(per_sweep).reshape(-1, 7).mean(axis=1)
    assert r["chunks_done"] == len(chunks) and 2 <= r["chunks_done"] <= 6
    assert abs(r["mean_par_last"] - chunks[-1]) < 1e-15 and abs(r["mean_par_prev"] - chunks[-2]) < 1e-15
    d = np.abs(np.diff(chunks))
    if r["converged"]:
        assert d[-1] <= 1e-4 and np.all(d[:-1] > 1e-4)          # the first acceptable pair stops the step
    else:
        assert r["chunks_done"] == 6 and np.all(d > 1e-4)
    # a huge threshold accepts after exactly min_chunks, a zero threshold never accepts
    _, o3 = _relax_case()
    r3 = o3.relax((1.0, 0.0, 0.0), chunk_sweeps=3, min_chunks=3, max_chunks=9, threshold=10.0)
    assert r3["converged"] and r3["chunks_done"] == 3 and r3["sweeps"] == 9
    _, o4 = _relax_case()
    r4 = o4.relax((1.0, 0.0, 0.0), chunk_sweeps=2, min_chunks=2, max_chunks=4, threshold=0.0)
    assert (not r4["converged"]) and r4["chunks_done"] == 4
    # the direction is normalised: (2, 0, 0) and (1, 0, 0) give the same projection
    _, o5 = _relax_case()
    r5 = o5.relax((2.0, 0.0, 0.0), chunk_sweeps=7, min_chunks=2, max_chunks=6, threshold=1e-4)
    assert r5["chunks_done"] == r["chunks_done"] and abs(r5["mean_par_last"] - r["mean_par_last"]) < 1e-15


# ------------------------------------------------------------------------------------------------ histograms
def test_histograms_against_numpy_and_closed_forms():
    """The oracle's length / angle histograms pinned against numpy.histogram (a library routine with its own edge logic) on
    states without values on bin edges, against hand-placed vectors with known angles to the mean direction, and against
    the totals."""
    import workloads as W
    wl = W.cfg5(nx=160, ny=150)                      # empty cells present
    o = O.OracleMMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, store_fp32=True)
    W.configure(o, wl, O.Material)
    rng = np.random.default_rng(5)
    v = rng.normal(size=(3, wl.N)); v /= np.linalg.norm(v, axis=0)
    v[2] = np.abs(v[2]) + 0.3                        # a clear mean direction
    o.set_m(*(rng.uniform(0.2, 0.9, wl.N) * v).astype(np.float32))
    ms = np.array([r["Ms0"] for r in wl.regions])[wl.region_of_cell] > 0
    m = np.stack([np.asarray(o.m[a], dtype=np.float64)[ms] for a in range(3)])
    L = np.linalg.norm(m, axis=0)
    c, u, ov = o.histogram("length", 100, 0.25, 0.8)
    ref, _ = np.histogram(L, bins=100, range=(0.25, 0.8))
    assert np.array_equal(c.astype(np.int64), ref - np.bincount([99], minlength=100) * np.count_nonzero(L == 0.8))
    assert u == np.count_nonzero(L < 0.25) and ov == np.count_nonzero(L >= 0.8) and c.sum() + u + ov == ms.sum() > 1000
    d = m.sum(axis=1); d /= np.linalg.norm(d)
    th = np.arccos(np.clip(m.T @ d / L, -1, 1))
    c2, u2, ov2 = o.histogram("angle", 100, th.min(), th.max() * (1 + 1e-12))       # the paper's range: min .. max theta
    ref2, _ = np.histogram(th, bins=100, range=(th.min(), th.max() * (1 + 1e-12)))
    assert np.array_equal(c2.astype(np.int64), ref2) and u2 == 0 and ov2 == 0
    # hand-placed: 3 vectors at polar angle 30 deg around z with azimuths 0, 120, 240 deg (mean direction = z exactly by
    # symmetry) and one along z: angles 30, 30, 30, 0 degrees
    o2 = O.OracleMMC(2, 2, 1, 5e-9, 5e-9, 5e-9, 0, store_fp32=False)
    o2.set_material([O.Material(Ms0=8e5, A0=1e-11, Tc=800.0)], None); o2.set_temperature(300.0, None)
    s, cth = np.sin(np.pi / 6), np.cos(np.pi / 6)
    az = np.array([0.0, 2 * np.pi / 3, 4 * np.pi / 3])
    o2.set_m(np.append(0.5 * s * np.cos(az), 0.0), np.append(0.5 * s * np.sin(az), 0.0), np.append(0.5 * cth * np.ones(3), 0.7))
    c3, u3, ov3 = o2.histogram("angle", 18, 0.0, np.pi)                              # 10-degree bins
    expect = np.zeros(18, dtype=np.uint64); expect[0] = 1
    third = o2.histogram("angle", 180, 0.0, np.pi)[0]                                # 1-degree bins: 30 deg sits on an edge
    assert c3[0] == 1 and c3[2] + c3[3] == 3 and c3.sum() == 4 and u3 == 0 and ov3 == 0
    assert third[0] == 1 and third[29] + third[30] == 3
    cl, _, _ = o2.histogram("length", 4, 0.35, 0.75)                                  # lengths 0.5, 0.5, 0.5, 0.7
    assert list(cl) == [0, 3, 0, 1]


# ------------------------------------------------------------------------------------------------ cubic anisotropy, Eq. (12)
def _cubic_cell(K1c, K2c, axes=((1, 0, 0), (0, 1, 0)), T=300.0, Tc=1044.0):
    s = O.OracleMMC(2, 2, 1, 5e-9, 5e-9, 5e-9, 0, store_fp32=False)
    (a, b) = axes
    s.set_material([O.Material(Ms0=1.71e6, A0=0.0, Tc=Tc, K1c=K1c, K2c=K2c, c1x=a[0], c1y=a[1], c1z=a[2], c2x=b[0], c2y=b[1], c2z=b[2])], None)
    s.set_temperature(T, None)
    return s


def test_cubic_anisotropy_textbook_values_symmetry_and_scaling():
    """Eq. (12) against what the mathematics fixes: the textbook energies of the principal directions
    (<100>: 0, <110>: K1/4, <111>: K1/3 + K2/27), invariance under the cubic group and under a common rotation of axes and
    vector, independence of |m| ("direction cosines"), the me^10 / me^21 temperature scaling of PAPER.md:143, and
    local dF == difference of the read-out energy."""
    V = (5e-9) ** 3
    me = O.me_of_T(300.0, 1044.0)
    for K1c, K2c in ((4.8e4, 0.0), (0.0, -1e4), (4.8e4, -1e4)):
        s = _cubic_cell(K1c, K2c)
        def E(v):
            s.set_m(*[np.full(4, x, dtype=np.float64) for x in v]); return s.observables()["E_an"] / 4
        k1, k2 = K1c * me ** 10, K2c * me ** 21
        assert E((0.7, 0, 0)) == pytest.approx(0.0, abs=1e-40)
        assert E((0.5, 0.5, 0)) == pytest.approx(V * k1 / 4, rel=1e-12)
        assert E((0.3, 0.3, 0.3)) == pytest.approx(V * (k1 / 3 + k2 / 27), rel=1e-12)
        v = np.array([0.31, -0.52, 0.77])
        e0 = E(v)
        assert E(2.5 * v) == pytest.approx(e0, rel=1e-12)                         # direction only
        for perm in ((1, 0, 2), (2, 1, 0), (1, 2, 0)):
            for sg in ((1, 1, 1), (-1, 1, 1), (1, -1, -1)):
                assert E(np.array(sg) * v[list(perm)]) == pytest.approx(e0, rel=1e-12)
    # common rotation of the axes and the vector
    rng = np.random.default_rng(3)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    s0 = _cubic_cell(4.8e4, -1e4); s1 = _cubic_cell(4.8e4, -1e4, axes=(Q[:, 0], Q[:, 1] + 0.3 * Q[:, 0]))   # Gram-Schmidt removes the 0.3
    v = np.array([0.31, -0.52, 0.77]); w = Q @ v * np.linalg.det(np.column_stack([Q[:, 0], Q[:, 1], np.cross(Q[:, 0], Q[:, 1])]))
    s0.set_m(*[np.full(4, x) for x in v]); s1.set_m(*[np.full(4, x) for x in (Q @ v)])
    assert s1.observables()["E_an"] == pytest.approx(s0.observables()["E_an"], rel=1e-12)
    # temperature scaling: K1 ~ me^10, K2 ~ me^21; zero at and above Tc
    for K1c, K2c, power in ((4.8e4, 0.0, 10), (0.0, -1e4, 21)):
        Es = []
        for T in (300.0, 800.0):
            s = _cubic_cell(K1c, K2c, T=T); s.set_m(*[np.full(4, x) for x in (0.3, 0.3, 0.3)]); Es.append(s.observables()["E_an"])
        assert Es[1] / Es[0] == pytest.approx((O.me_of_T(800.0, 1044.0) / me) ** power, rel=1e-10)
    s = _cubic_cell(4.8e4, -1e4, T=1044.0); s.set_m(*[np.full(4, x) for x in (0.3, 0.3, 0.3)])
    assert s.observables()["E_an"] == 0.0
    # local dF = difference of the read-out, in units of kB T
    s = _cubic_cell(4.8e4, -1e4)
    m0 = np.array([0.5, 0.2, -0.4]); s.set_m(*[np.full(4, x) for x in m0])
    dm = np.array([-0.1, 0.25, 0.05])
    eb = s.observables()["E_an"]; t = s.cell_dF(1, 0, 0, dm)
    s.m[0][1] += dm[0]; s.m[1][1] += dm[1]; s.m[2][1] += dm[2]
    assert t[1] * KB * 300.0 == pytest.approx(s.observables()["E_an"] - eb, rel=1e-10)


def test_cubic_anisotropy_single_cell_distribution():
    """Fixed-length cells with cubic anisotropy only sample exp(-V K1(T) c1(n) / kT) uniformly in solid angle (Eq. (6),
    reading G6): <c1> against a plain quadrature over the sphere; K1 > 0 favours <100>, so <c1> lies below the isotropic 1/5."""
    T, Tc, L = 300.0, 1044.0, 0.9
    V = (8e-9) ** 3
    s = O.OracleMMC(24, 24, 1, 8e-9, 8e-9, 8e-9, 0b011, store_fp32=False)
    s.set_material([O.Material(Ms0=1.71e6, A0=0.0, Tc=Tc, K1c=2.0e5, K2c=0.0)], None)
    s.set_temperature(T, None); s.set_move(40.0, 0.0, False); s.set_seed(12)
    rng = np.random.default_rng(8)
    v = rng.normal(size=(3, 576)); v /= np.linalg.norm(v, axis=0)
    s.set_m(*(L * v))
    s.run(300)
    acc = 0.0; n = 0
    for _ in range(120):
        s.run(5)
        a, b, g = (s.m[q] / L for q in range(3))
        acc += (a * a * b * b + a * a * g * g + b * b * g * g).mean(); n += 1
    kappa = V * 2.0e5 * O.me_of_T(T, Tc) ** 10 / (KB * T)
    th = np.linspace(0, np.pi, 1201); ph = np.linspace(0, 2 * np.pi, 2401)
    TH, PH = np.meshgrid(th, ph, indexing="ij")
    x, y, z = np.sin(TH) * np.cos(PH), np.sin(TH) * np.sin(PH), np.cos(TH)
    c1 = x * x * y * y + x * x * z * z + y * y * z * z
    w = np.exp(-kappa * c1) * np.sin(TH)
    expect = np.trapezoid(np.trapezoid(c1 * w, ph, axis=1), th) / np.trapezoid(np.trapezoid(w, ph, axis=1), th)
    assert kappa > 1.0 and expect < 0.19
    assert acc / n == pytest.approx(expect, rel=2e-2)


def test_uniaxial_k2_term_of_eq11():
    """Second term of Eq. (11) (reading G5: m_i = m/me, both terms times V, K2(T) = K2 me^10): the textbook
    K2 sin^4(theta) for a vector of the equilibrium length at polar angle theta to the axis, zero along the axis, the me^10
    temperature scaling, zero at Tc, and local dF == difference of the read-out."""
    V = (5e-9) ** 3
    def cell(T, K1=0.0, K2=2e5):
        s = O.OracleMMC(2, 2, 1, 5e-9, 5e-9, 5e-9, 0, store_fp32=False)
        s.set_material([O.Material(Ms0=8e5, A0=0.0, K1=K1, K2=K2, ax=0.0, ay=0.6, az=0.8, Tc=870.0)], None)
        s.set_temperature(T, None)
        return s
    me = O.me_of_T(300.0, 870.0)
    s = cell(300.0)
    e = np.array([0.0, 0.6, 0.8]); perp = np.array([1.0, 0.0, 0.0])
    for th in (0.0, 0.3, 1.0, np.pi / 2):
        v = me * (np.cos(th) * e + np.sin(th) * perp)
        s.set_m(*[np.full(4, x) for x in v])
        assert s.observables()["E_an"] / 4 == pytest.approx(V * 2e5 * me ** 10 * np.sin(th) ** 4, rel=3e-6, abs=1e-30)   # the state is stored in fp32
    # temperature scaling and T = Tc
    v = np.array([0.4, 0.1, 0.2])
    Es = []
    for T in (300.0, 700.0):
        s = cell(T); s.set_m(*[np.full(4, x) for x in v]); Es.append(s.observables()["E_an"])
    m3, m7 = O.me_of_T(300.0, 870.0), O.me_of_T(700.0, 870.0)
    g = lambda me_: (1 - (v @ e) ** 2 / me_ ** 2) ** 2 * me_ ** 10
    assert Es[1] / Es[0] == pytest.approx(g(m7) / g(m3), rel=3e-6)
    s = cell(870.0); s.set_m(*[np.full(4, x) for x in v]); assert s.observables()["E_an"] == 0.0
    # local dF (K1 and K2 together) = difference of the read-out
    s = cell(300.0, K1=5e5)
    s.set_m(*[np.full(4, x) for x in v])
    dm = np.array([0.05, -0.2, 0.1])
    eb = s.observables()["E_an"]; t = s.cell_dF(0, 1, 0, dm)
    for a in range(3):
        s.m[a][2] += dm[a]
    assert t[1] * KB * 300.0 == pytest.approx(s.observables()["E_an"] - eb, rel=1e-10)


def test_uniaxial_k1_readout_constant_is_textbook_k1_sin2():
    """First term of Eq. (11) in the read-out (reading G5): E_an = V K1(T) [1 - (m.e)^2/me^2] with
    K1(T) = K1 me^3 (l = 2), i.e. the textbook K1(T) sin^2(theta) for a vector of the equilibrium length at
    polar angle theta to the axis -- in particular exactly zero along the axis, which pins the constant V K1 me^3 that no
    energy DIFFERENCE can see -- and zero at and above Tc."""
    V = (5e-9) ** 3
    e = np.array([0.0, 0.6, 0.8]); perp = np.array([1.0, 0.0, 0.0])
    for T in (300.0, 700.0):
        me = O.me_of_T(T, 870.0)
        s = O.OracleMMC(2, 2, 1, 5e-9, 5e-9, 5e-9, 0, store_fp32=False)
        s.set_material([O.Material(Ms0=8e5, A0=0.0, K1=5e5, ax=0.0, ay=0.6, az=0.8, Tc=870.0)], None)
        s.set_temperature(T, None)
        for th in (0.0, 0.4, 1.1, np.pi / 2, 2.5):
            v = me * (np.cos(th) * e + np.sin(th) * perp)
            s.m = [np.full(4, x) for x in v]                       # fp64 state: no storage rounding in this pin
            assert s.observables()["E_an"] / 4 == pytest.approx(V * 5e5 * me ** 3 * np.sin(th) ** 2, rel=1e-12, abs=1e-12 * V * 5e5)
    s = O.OracleMMC(2, 2, 1, 5e-9, 5e-9, 5e-9, 0, store_fp32=False)
    s.set_material([O.Material(Ms0=8e5, A0=0.0, K1=5e5, ax=0.0, ay=0.6, az=0.8, Tc=870.0)], None)
    for T in (870.0, 900.0):
        s.set_temperature(T, None); s.m = [np.full(4, x) for x in (0.02, 0.01, 0.03)]
        assert s.observables()["E_an"] == 0.0
