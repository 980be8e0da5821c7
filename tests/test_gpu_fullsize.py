"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (production kernels through
mmc_sweep / mmc_demag_field, not the debug pass), plus the equilibrium 3-sigma checks of north_star.

  demag   sampled outputs the oracle computes one by one: B_d(r_i) = -mu0 sum_j N(r_i - r_j) M_j (Eq. (14),
          PAPER.md:120) as a direct sum over the oracle's own tensor table, at cells spread over the mesh
          (corners, edges, centre, random); bar 2e-5 max|B| as in test_gpu_parity.
  sweep   one whole iteration of mmc_sweep on the full mesh against the oracle's red + black passes on the same
          state and Philox stream, each side with its own demag field; bar as in
          test_sweep_matches_replayed_oracle: all cells equal to 2e-6 except a 2e-3 fraction (near-margin decisions
          and their black neighbours).
  equilibrium  8 seeds on each side, blocked means after discarding the first half, Welch test at 3 sigma.
  paper       the length distribution of the CUDA path itself against the exact chain means derived from Eq. (7)
              (tests/golden/length_means.txt), five temperatures below, at and above Tc, two sigma.
"""
import numpy as np
import pytest

import oracle as O
import workloads as W

pytestmark = pytest.mark.gpu

MU0 = 4e-7 * np.pi


def _np(ts):
    return [t.detach().cpu().numpy().astype(np.float64) for t in ts]


def _gpu(wl):
    import paper_2106_05593_b200 as P
    s = P.MMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask)
    W.configure(s, wl, P.Material)
    return s


def _orc(wl):
    s = O.OracleMMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, store_fp32=True)
    W.configure(s, wl, O.Material)
    return s


_CONV = {}


def _conv(cfg, wl):
    """The oracle's fp64 FFT convolution object (tensor table + spectrum) of a config, built once per session."""
    if cfg not in _CONV:
        _CONV[cfg] = O.DemagFFT(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz)
    return _CONV[cfg]


def _ms0_of_cell(wl):
    ms = np.array([r["Ms0"] for r in wl.regions], dtype=np.float64)
    if wl.region_of_cell is None:
        return np.full(wl.N, ms[0])
    return ms[wl.region_of_cell]


def _direct_sample(tab, M, i, j, k):
    """Eq. (14) at one cell: the octant table holds N(|ox|,|oy|,|oz|); diagonal components are even in every coordinate,
    N_ab (a != b) is odd in coordinates a and b."""
    _, nz, ny, nx = tab.shape
    ox = i - np.arange(nx); oy = j - np.arange(ny); oz = k - np.arange(nz)
    ax, ay, az = np.abs(ox), np.abs(oy), np.abs(oz)
    sx, sy, sz = np.sign(ox), np.sign(oy), np.sign(oz)
    sub = [tab[q][np.ix_(az, ay, ax)] for q in range(6)]
    SX = sx[None, None, :]; SY = sy[None, :, None]; SZ = sz[:, None, None]
    xx, yy, zz = sub[0], sub[1], sub[2]
    xy = sub[3] * SX * SY; xz = sub[4] * SX * SZ; yz = sub[5] * SY * SZ
    Mx, My, Mz = M
    hx = -(xx * Mx + xy * My + xz * Mz).sum()
    hy = -(xy * Mx + yy * My + yz * Mz).sum()
    hz = -(xz * Mx + yz * My + zz * Mz).sum()
    return MU0 * np.array([hx, hy, hz])


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_demag_sampled(cfg):
    wl = W.make(cfg)
    g = _gpu(wl)
    bg = _np(g.demag_field())
    g.close()
    nx, ny, nz = wl.nx, wl.ny, wl.nz
    tab = _conv(cfg, wl).tab
    ms0 = _ms0_of_cell(wl)
    M = [(ms0 * wl.m0[a].astype(np.float64)).reshape(nz, ny, nx) for a in range(3)]
    rng = np.random.default_rng(1000 + cfg)
    pts = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (nx - 1, 0, 0), (0, ny - 1, nz - 1), (nx // 2, ny // 2, nz // 2),
           (nx // 2 - 1, 0, 0), (1, ny // 2, nz - 1), (nx - 2, ny - 3, 0)]
    pts += [(int(rng.integers(nx)), int(rng.integers(ny)), int(rng.integers(nz))) for _ in range(16)]
    worst = scale = 0.0                       # scale = max |B| over the oracle's own samples (corners and edges included)
    for (i, j, k) in pts:
        bo = _direct_sample(tab, M, i, j, k)
        c = i + nx * (j + ny * k)
        worst = max(worst, max(abs(bg[a][c] - bo[a]) for a in range(3)))
        scale = max(scale, np.abs(bo).max())
    assert worst <= 2e-5 * scale, f"cfg{cfg}: worst sampled |B_gpu - B_direct| = {worst:.3e} T vs scale {scale:.3e} T"


def _full_iteration(cfg, updates):
    from parity_util import explain_iteration
    wl = W.make(cfg)
    wl.adaptive_cone = False
    g, o = _gpu(wl), _orc(wl)
    if wl.demag:
        o._demag = _conv(cfg, wl)             # the oracle's own field (numpy.fft on the padded grid), nothing from the GPU
        g.set_demag(True, updates); o.set_demag(True, updates)
    g.sweep(1)
    mg = _np(g.get_m())
    r = explain_iteration(wl, o, mg)
    label = f"cfg{cfg}, {updates} field update(s)"
    print(f"{label}: {r['flips']} decision flips among {r['active']} trials, {r['unexplained']} unexplained")
    assert r["untouched_ok"], f"{label}: a cell without a trial changed"
    assert r["neither"] == 0, f"{label}: {r['neither']} cells hold neither the accepted nor the rejected candidate"
    assert r["unexplained"] == 0, f"{label}: {r['unexplained']} of {r['flips']} flips are not explained by the oracle's margins"
    assert r["flips"] <= max(2, 2e-3 * wl.n_active), f"{label}: {r['flips']} of {wl.n_active} decisions differ"
    ob = g.observables()
    assert ob["sweeps_done"] == 1 and ob["trials"] == wl.n_active == r["active"]
    assert abs(int(ob["accepted"]) - r["oracle_accepted"]) <= r["flips"]
    # empty cells are never touched
    if wl.n_active < wl.N:
        empty = _ms0_of_cell(wl) == 0
        for a in range(3):
            assert np.array_equal(mg[a][empty], wl.m0[a][empty].astype(np.float64))
    g.close()


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_sweep(cfg):
    """One whole iteration at full size in the production launch configuration.  Every active cell must hold the oracle's
    accepted or rejected candidate; every decision that differs must lie inside the oracle's own margin window (or be a
    black neighbour of such a red cell): a defect confined to one face or tile of the launch geometry cannot hide in a
    count (tests/parity_util.py)."""
    _full_iteration(cfg, 1)


@pytest.mark.parametrize("cfg", [2, 4])
def test_full_size_sweep_two_field_updates(cfg):
    """The same with the field updated before each colour pass."""
    _full_iteration(cfg, 2)


# ------------------------------------------------------------------------------------------------ equilibrium, 3 sigma
def _series_gpu(wl, seed, n_sweeps):
    wl.seed = seed
    g = _gpu(wl)
    g.sweep(n_sweeps // 2)
    g.reset_averages(); g.reset_counters()
    g.sweep(n_sweeps - n_sweeps // 2)
    ob = g.observables()
    g.close()
    e = sum(ob[k] for k in ("E_ex", "E_an", "E_zee", "E_dmi", "E_demag", "E_long")) / wl.n_active
    return np.array([ob["run_mean_len"], ob["run_mean_m"][2], ob["accepted"] / ob["trials"], ob["run_mean_m"][0], e / _KT_REF])


def _series_oracle(wl, seed, n_sweeps):
    wl.seed = seed
    o = _orc(wl)
    o.run(n_sweeps // 2)
    acc0, tri0 = o.accepted, o.trials
    s_len = s_mz = s_mx = 0.0
    n2 = n_sweeps - n_sweeps // 2
    act = _ms0_of_cell(wl) > 0
    for _ in range(n2):
        o.run(1)
        s_len += np.sqrt(o.m[0] ** 2 + o.m[1] ** 2 + o.m[2] ** 2)[act].mean()
        s_mz += o.m[2][act].mean(); s_mx += o.m[0][act].mean()
    ob = o.observables()
    e = sum(ob[k] for k in ("E_ex", "E_an", "E_zee", "E_dmi", "E_demag", "E_long")) / wl.n_active
    return np.array([s_len / n2, s_mz / n2, (o.accepted - acc0) / (o.trials - tri0), s_mx / n2, e / _KT_REF])


_KT_REF = 1.380649e-23 * 300.0      # energies per cell are compared in units of kB x 300 K

EQ_CASES = {
    # permalloy film with demag in a field along x (the hysteresis config), open boundaries
    "cfg2_32x32": (lambda: W.cfg2(nx=32, ny=32), 1500),
    # artificial spin ice: empty cells, islands, field along [11]
    "cfg5_140x140": (lambda: W.cfg5(nx=140, ny=140), 400),
    # exchange + uniaxial anisotropy, paper regime (acceptance ~ 0.5), far below Tc
    "cfg1_paper_regime_32x32": (lambda: W.cfg1(paper_regime=True), 4000),
    # BASELINE.json config 1 exactly as written: sigma = 0.05, cone 30 deg fixed, 1000 sweeps (acceptance ~1 %)
    "cfg1_as_written_32x32": (lambda: W.cfg1(), 1000),
    # chiral film just below Tc (650 K of Tc 700 K): exchange + DMI + anisotropy + Zeeman + demag + wide length distribution
    "cfg3_32x32_650K": (lambda: W.cfg3(nx=32, ny=32, T=650.0), 3000),
    # granular film: per-cell classes, grain boundaries, hot spot above Tc, 3 layers, demag
    "cfg4_24x24x3": (lambda: W.cfg4(nx=24, ny=24, nz=3), 2000),
    # granular Fe film: cubic anisotropy (Eq. (12)) with random axes per grain, periodic in the plane, demag
    "fe_film_cubic_24x24x3": (lambda: W.fe_film(nx=24, ny=24, nz=3), 2000),
}


@pytest.mark.parametrize("name", list(EQ_CASES))
def test_equilibrium_observables_within_3_sigma(name):
    """north_star: equilibrium observables within 3 sigma.  8 independent Philox keys per side (different keys on the
    two sides, so this is a statistical comparison, not a replay); per-run means of <|m|>, <m_z>, <m_x> and the acceptance
    rate over the second half of the run, and the total energy per cell of the final state; Welch statistic
    |mean_g - mean_o| <= 3 sqrt(var_g/8 + var_o/8)."""
    make, n_sweeps = EQ_CASES[name]
    G = np.array([_series_gpu(make(), 7000 + s, n_sweeps) for s in range(8)])
    Oo = np.array([_series_oracle(make(), 9000 + s, n_sweeps) for s in range(8)])
    for q, label in enumerate(("mean |m|", "mean m_z", "acceptance", "mean m_x", "energy per cell / kB 300 K")):
        mg, mo = G[:, q].mean(), Oo[:, q].mean()
        se = np.sqrt(G[:, q].var(ddof=1) / 8 + Oo[:, q].var(ddof=1) / 8)
        assert abs(mg - mo) <= 3.0 * se + 1e-7 + 2e-6 * abs(mo), f"{name}: {label}: gpu {mg:.6f} vs oracle {mo:.6f}, 3 sigma = {3 * se:.2e}"


# ------------------------------------------------------------------------------------------------ the CUDA path against the paper's distribution
def _golden_rows():
    import os
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "length_means.txt")) as f:
        for ln in f:
            if ln.strip() and not ln.startswith("#"):
                rows.append([float(x) for x in ln.split()])
    return rows


@pytest.mark.parametrize("sigma_col", [(0.03, 2), (0.05, 3)], ids=["sigma0.03", "sigma0.05"])
@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"T{int(r[0])}")
def test_gpu_length_distribution_matches_eq7_chain(row, sigma_col):
    """PAPER.md:108 / Eq. (7) on the CUDA path itself, against values that come from the paper and not from the oracle:
    1 048 576 decoupled cells (A0 = 0, no anisotropy, no field, no demag: an ensemble of single-cell chains) at the
    paper's Fig. 1 parameters (Tc 680 K, V = (5 nm)^3, Ms0 8e5 A/m, mu_B), 20 000 iterations of burn-in from a spread of
    lengths and 20 000 of averaging (the length walk near Tc decorrelates over thousands of iterations).  The running
    mean of |m| must hit the exact stationary mean of the literal (m_B/m_A)^4 chain (tests/golden/length_means.txt,
    SURVEY 8(c) G1; T = 680 K is the T = Tc limit of G10) to 5e-4 relative (measured: 3e-5 .. 1.3e-4) -- which tells
    sigma = 0.03 from 0.05 (1.6e-3 .. 3e-3 apart) and the chain from the Eq. (7) quadrature mean (2.4e-3 .. 8e-3 below it,
    the bias linear in sigma of reading G1)."""
    import paper_2106_05593_b200 as P
    sigma, col = sigma_col
    T, m7, ref = row[0], row[1], row[col]
    n = 1024
    rng = np.random.default_rng(int(T))
    v = rng.normal(size=(3, n * n)); v /= np.linalg.norm(v, axis=0)
    m0 = (row[2] * rng.uniform(0.3, 1.7, n * n) * v).astype(np.float32)
    g = P.MMC(n, n, 1, 5e-9, 5e-9, 5e-9, 0b011)
    g.set_material([P.Material(Ms0=8e5, A0=0.0, K1=0.0, Tc=680.0)])
    g.set_temperature(T); g.set_field(0.0, 0.0, 0.0); g.set_move(60.0, sigma, False); g.set_demag(False)
    g.set_seed(680000 + int(T)); g.set_m(*m0)
    g.sweep(20000)
    g.reset_averages()
    g.sweep(20000)
    ob = g.observables()
    g.close()
    assert ob["run_mean_len"] == pytest.approx(ref, rel=5e-4)
    assert ob["run_mean_len"] > m7 * (1.0 + 1.5e-3)


def test_gpu_angular_distribution_is_langevin():
    """Transverse part of the distribution (Eq. (6), :114) on the CUDA path against the closed form: decoupled
    cells of fixed length (sigma = 0: the move is a pure cone rotation) in a field along z sample exp(xi cos(theta)) uniformly in
    solid angle (reading G6), so <cos(theta)> = coth(xi) - 1/xi with xi = V Ms0 |m| B / kB T."""
    import paper_2106_05593_b200 as P
    kB = 1.380649e-23
    T, V, Ms0, L = 300.0, (5e-9) ** 3, 8e5, 0.9
    for xi in (0.5, 3.0, 12.0):
        B = xi * kB * T / (V * Ms0 * L)
        n = 512
        rng = np.random.default_rng(int(10 * xi))
        v = rng.normal(size=(3, n * n)); v /= np.linalg.norm(v, axis=0)
        m0 = (L * v).astype(np.float32)
        g = P.MMC(n, n, 1, 5e-9, 5e-9, 5e-9, 0b011)
        g.set_material([P.Material(Ms0=Ms0, A0=0.0, K1=0.0, Tc=680.0)])
        g.set_temperature(T); g.set_field(0.0, 0.0, B); g.set_move(50.0, 0.0, False); g.set_demag(False)
        g.set_seed(int(1000 * xi)); g.set_m(*m0)
        g.sweep(1500); g.reset_averages(); g.sweep(3000)
        ob = g.observables()
        g.close()
        assert ob["run_mean_len"] == pytest.approx(L, rel=2e-6)                 # rotations keep the length
        expect = 1.0 / np.tanh(xi) - 1.0 / xi
        assert ob["run_mean_m"][2] / L == pytest.approx(expect, abs=3e-4), f"xi = {xi}"
        assert abs(ob["run_mean_m"][0]) < 3e-4 and abs(ob["run_mean_m"][1]) < 3e-4


# ------------------------------------------------------------------------------------------------ whole schedules (soak)
def test_cfg2_hysteresis_branch_full_size():
    """BASELINE.json config 2 as written: 256x256x1 permalloy film, demag, B_x from +100 mT to -100 mT in 2 mT steps, 200
    iterations per step (20 200 iterations with the adaptive cone).  Sanity of the physics over a long run: the film starts
    and ends saturated along the field, the branch is monotone within noise, reverses in one piece, |m| stays at me(300 K), the
    acceptance rate is held near 0.5 by the cone controller, nothing leaves the physical range."""
    import paper_2106_05593_b200 as P
    from paper_2106_05593_b200.schedule import run_schedule
    wl = W.make(2)
    g = _gpu(wl)
    rows = run_schedule(g, wl)
    mx = np.array([r["mean_m"][0] for r in rows]); ml = np.array([r["mean_len"] for r in rows])
    assert len(rows) == 101 and g.observables()["sweeps_done"] == 20200
    assert mx[0] > 0.8 and mx[-1] < -0.5                              # 200 iterations per step: the reversal is under way, not complete
    assert np.all(np.diff(mx) < 5e-3)                                  # decreasing field: m_x never climbs back
    assert np.all(np.abs(ml - 0.8675) < 2e-3) and np.all(np.isfinite(mx))
    acc = np.array([r["acceptance"] for r in rows[20:]])
    assert np.all((acc > 0.35) & (acc < 0.65))
    m = _np(g.get_m())
    L = np.sqrt(m[0] ** 2 + m[1] ** 2 + m[2] ** 2)
    assert L.max() < 1.0 and L.min() > 0.5
    g.close()


def test_cfg3_temperature_sweep_tracks_the_length_curve():
    """BASELINE.json config 3 (reduced to 128x128 and 1000 iterations per temperature): T from 200 K to 800 K through Tc = 700 K
    with the state carried over.  <|m|> follows me(T) far below Tc, stays ABOVE me near and above Tc (the mean
    of the length distribution is not me), decreases monotonically, and the T = Tc step (reading G10) runs."""
    from paper_2106_05593_b200.schedule import run_schedule
    wl = W.cfg3(nx=128, ny=128)
    wl.schedule = [("T", T, 1000) for (_, T, _) in wl.schedule]
    g = _gpu(wl)
    rows = run_schedule(g, wl)
    T = np.array([r["value"] for r in rows]); ml = np.array([r["mean_len"] for r in rows])
    assert 700.0 in T and T[0] == 200.0 and T[-1] == 800.0
    assert np.all(np.diff(ml) < 0)
    me = np.array([O.me_of_T(float(t), 700.0) for t in T])
    assert abs(ml[0] - me[0]) < 2e-3                                   # 200 K: the chain sits at me
    assert np.all(ml[T >= 650.0] > me[T >= 650.0] + 0.01)              # near and above Tc: mean length > me (0 above Tc)
    assert ml[-1] < 0.2                                                # 800 K, 2 nm cells: a broad distribution around 0.14
    g.close()
