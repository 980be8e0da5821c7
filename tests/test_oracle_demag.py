"""Pins of the oracle's demagnetising path (Eq. (14))."""
import os

import numpy as np
import pytest

import oracle as O

KB = 1.380649e-23

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def test_newell_probe_values():
    for r in _rows("newell_probe.txt"):
        v = [float(x) for x in r]
        assert np.allclose(O.newell(*v[:6]), v[6:12], rtol=2e-11, atol=1e-15)


def test_newell_trace_and_symmetry():
    """Self term of a cube = 1/3 each, trace 1 at the origin and 0 elsewhere (div B = 0); off-diagonals vanish on
    the coordinate planes; diagonal components even, N_ab odd in a and b."""
    d = (1.0, 0.7, 1.9)
    n0 = O.newell(0, 0, 0, *d)
    assert n0[:3].sum() == pytest.approx(1.0, abs=1e-15) and np.all(np.abs(n0[3:]) < 1e-30)
    assert np.allclose(O.newell(0, 0, 0, 2, 2, 2)[:3], 1 / 3, atol=1e-16)
    rng = np.random.default_rng(0)
    for _ in range(20):
        o = rng.integers(-6, 7, 3)
        if not o.any():
            continue
        X, Y, Z = o * np.array(d)
        n = O.newell(X, Y, Z, *d)
        assert abs(n[:3].sum()) < 1e-16
        nm = O.newell(-X, Y, Z, *d)
        assert np.allclose(nm, n * np.array([1, 1, 1, -1, -1, 1]), rtol=1e-13, atol=1e-30)
        if o[2] == 0:
            assert abs(n[4]) < 1e-30 and abs(n[5]) < 1e-30            # N_xz = N_yz = 0 at Z = 0


def _quad_tensor(R, d, n=10):
    """Independent definition: N_ab(R) = (1/V) int_cell int_cell K_ab(R + u - v) du dv,
    K_ab = (1/4 pi)(delta_ab/r^3 - 3 r_a r_b/r^5); u - v has a triangular weight (d - |w|) per axis;
    Gauss-Legendre on [-d, 0] and [0, d]."""
    x, w = np.polynomial.legendre.leggauss(n)
    axes = []
    for da in d:
        pts = np.concatenate([-da / 2 + da / 2 * x, da / 2 + da / 2 * x])
        wts = np.concatenate([w, w]) * da / 2 * (da - np.abs(pts))
        axes.append((pts, wts))
    WX, WY, WZ = np.meshgrid(axes[0][0], axes[1][0], axes[2][0], indexing="ij")
    wt = axes[0][1][:, None, None] * axes[1][1][None, :, None] * axes[2][1][None, None, :]
    rx, ry, rz = R[0] + WX, R[1] + WY, R[2] + WZ
    r2 = rx * rx + ry * ry + rz * rz; r5 = r2 ** 2.5
    V = d[0] * d[1] * d[2]
    f = lambda a, b, dl: ((dl * r2 - 3 * a * b) / r5 * wt).sum() / (4 * np.pi * V)
    return np.array([f(rx, rx, 1), f(ry, ry, 1), f(rz, rz, 1), f(rx, ry, 0), f(rx, rz, 0), f(ry, rz, 0)])


@pytest.mark.parametrize("off,d", [((3, 2, 1), (1, 1, 1)), ((2, 0, 0), (1, 1, 1)), ((0, 2, 1), (1, 1, 1)),
                                   ((2, 1, 0), (1, 1, 2)), ((0, 0, 2), (1, 1, 2)), ((1, 2, 1), (1, 1, 2)),
                                   ((4, -3, 2), (5e-9, 4e-9, 3e-9))])
def test_newell_against_6d_quadrature(off, d):
    R = np.array(off, float) * np.array(d)
    ref = _quad_tensor(R, d, n=14)
    got = O.newell(*R, *d)
    assert np.allclose(got, ref, rtol=2e-7, atol=2e-9 * np.abs(ref).max())


def test_newell_composition_identity():
    """The mean of N over all cell pairs of a uniformly magnetised block equals the self term of the block taken
    as one big cell (SURVEY pin: two stacked cubes 1/3 - 0.135017180544 = 0.198316152789; 6x5x2 block)."""
    two = O.newell(0, 0, 0, 1, 1, 2)[2]
    assert two == pytest.approx(1 / 3 + O.newell(0, 0, 1, 1, 1, 1)[2], rel=1e-13)
    nx, ny, nz = 6, 5, 2
    acc = np.zeros(6)
    for ox in range(-nx + 1, nx):
        for oy in range(-ny + 1, ny):
            for oz in range(-nz + 1, nz):
                cnt = (nx - abs(ox)) * (ny - abs(oy)) * (nz - abs(oz))
                acc += cnt * O.newell(ox, oy, oz, 1, 1, 1)
    acc /= nx * ny * nz
    big = O.newell(0, 0, 0, nx, ny, nz)
    assert np.allclose(acc, big, rtol=1e-12, atol=1e-15)
    assert big[2] == pytest.approx(0.56805647309712, rel=1e-11)


@pytest.mark.parametrize("d", [(5e-9, 5e-9, 5e-9), (5e-9, 5e-9, 10e-9)])
def test_far_field_matches_newell_beyond_r_near(d):
    """Sub-cube dipole average (O7) vs the binary128 Newell value where the two are stitched."""
    tab_far = O.demag_tensor(40, 40, 3, *d, r_near=32)
    tab_all = O.demag_tensor(40, 40, 3, *d, r_near=1000)
    far = np.zeros((3, 40, 40), bool); far[:, 33:, :] = True; far[:, :, 33:] = True
    scale = np.abs(tab_all[:3][:, far]).max()
    assert np.abs(tab_far - tab_all)[:, far].max() < 3e-6 * scale
    assert np.array_equal(tab_far[:, ~far], tab_all[:, ~far])


@pytest.mark.parametrize("shape,d", [((8, 6, 1), (5e-9, 5e-9, 5e-9)), ((5, 4, 3), (3e-9, 3e-9, 3e-9)),
                                     ((6, 7, 1), (5e-9, 5e-9, 10e-9)), ((4, 4, 2), (2e-9, 3e-9, 4e-9))])
def test_fft_convolution_equals_direct_sum(shape, d):
    nx, ny, nz = shape
    rng = np.random.default_rng(nx * 100 + ny * 10 + nz)
    M = rng.normal(size=(3, nz, ny, nx)) * 8e5
    M[:, rng.uniform(size=(nz, ny, nx)) < 0.25] = 0.0                    # empty cells
    conv = O.DemagFFT(nx, ny, nz, *d)
    b_fft = conv.field(*M)
    b_dir = O.demag_direct(conv.tab, *M)
    scale = max(np.abs(b).max() for b in b_dir)
    for a in range(3):
        assert np.abs(b_fft[a] - b_dir[a]).max() < 1e-13 * scale
    # the spectrum of the tensor is real (even/odd-odd symmetry of N)
    assert np.abs(conv.Khat.imag).max() < 1e-13 * np.abs(conv.Khat.real).max()


def test_uniform_block_field_is_minus_block_tensor_times_M():
    """Thin-film limit check through the whole path: a uniformly magnetised 12x10x1 block of cubes has
    mean H_d = -N_block M with N_block the Newell self term of the 12x10x1 cuboid; for M || z this is the
    perpendicular-film shape anisotropy that Figs. 3-6 rely on."""
    nx, ny, nz, h = 12, 10, 1, 5e-9
    conv = O.DemagFFT(nx, ny, nz, h, h, h)
    Nblk = O.newell(0, 0, 0, nx * h, ny * h, nz * h)
    for a in range(3):
        M = np.zeros((3, nz, ny, nx)); M[a] = 8e5
        b = conv.field(*M)
        for q in range(3):
            expect = -O.MU0 * 8e5 * (Nblk[a] if q == a else 0.0)
            assert b[q].mean() == pytest.approx(expect, abs=1e-12 * O.MU0 * 8e5)
    assert Nblk[2] > 0.8 and Nblk[0] < 0.1


def test_oracle_sweep_uses_frozen_field_once_per_iteration():
    """field computed at the start of the iteration, not updated on accept; optional second
    update before the black pass (updates_per_sweep = 2)."""
    nx = ny = 8
    rng = np.random.default_rng(3)
    v = rng.normal(size=(3, nx * ny)); v /= np.linalg.norm(v, axis=0)
    out = {}
    for upd in (1, 2):
        s = O.OracleMMC(nx, ny, 1, 5e-9, 5e-9, 5e-9, pbc_mask=0)
        s.set_material([O.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)]); s.set_temperature(300.0)
        s.set_move(20.0, -1.0, False); s.set_demag(True, upd); s.set_seed(5)
        s.set_m(*(0.8675 * v).astype(np.float32))
        b0 = s.demag_field()
        s.sweep_once()
        out[upd] = np.stack(s.m)
        if upd == 1:
            assert all(np.array_equal(s.bd[a], b0[a]) for a in range(3))     # still the start-of-iteration field
        else:
            assert not np.array_equal(s.bd[0], b0[0])
    red = np.array([(c % nx + c // nx) % 2 == 0 for c in range(nx * ny)])
    assert np.array_equal(out[1][:, red], out[2][:, red])                    # red pass saw the same field


# ------------------------------------------------------------------------------------------------ serial mode with exact demag (Appendix B)
def _ellipse(nx, ny, seed, T=300.0, B=(0.015, 0.0, 0.0)):
    """The paper's Appendix-B shape in small: a permalloy ellipse of nx x ny 5 nm cells, H = 12 kA/m."""
    j, i = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    inside = ((i + 0.5 - nx / 2) / (nx / 2)) ** 2 + ((j + 0.5 - ny / 2) / (ny / 2)) ** 2 <= 1.0
    reg = inside.ravel().astype(np.int32)
    s = O.OracleMMC(nx, ny, 1, 5e-9, 5e-9, 5e-9, 0, store_fp32=False)
    s.set_material([O.Material(), O.Material(Ms0=8e5, A0=1.3e-11, Tc=870.0)], reg)
    s.set_temperature(T, None); s.set_field(*B); s.set_move(12.0, -1.0, False); s.set_demag(True); s.set_seed(seed)
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(3, nx * ny)); v[0] += 2.5; v /= np.linalg.norm(v, axis=0)
    s.set_m(*(0.86 * v * reg))
    return s, reg


def test_exact_demag_dF_is_the_global_energy_change():
    """PAPER.md:218 / SURVEY O8: for a single-cell move the exact change of E_d = (mu0 V/2) sum M_i N_ij M_j is the field term
    with the current field plus the self term (mu0 V/2) dM N(0) dM; checked against E_demag recomputed from scratch by the
    direct O(N^2) sum, while the frozen-field term of the parallel scheme misses exactly the self term."""
    s, reg = _ellipse(10, 6, 3)
    rng = np.random.default_rng(0)
    kT = KB * 300.0
    for c in np.flatnonzero(reg)[::7]:
        dm = rng.normal(size=3) * 0.2
        e0 = s.observables()["E_demag"]
        dF = s.exact_demag_dF(int(c), dm)
        for a in range(3):
            s.m[a][c] += dm[a]
        e1 = s.observables()["E_demag"]
        for a in range(3):
            s.m[a][c] -= dm[a]
        assert dF * kT == pytest.approx(e1 - e0, rel=1e-9, abs=1e-30)


def test_serial_exact_sweep_keeps_the_field_current():
    """After serial sweeps the incrementally updated field equals the field of the final state recomputed from scratch."""
    s, reg = _ellipse(12, 8, 5)
    b = s.run_serial_exact(3)
    assert s.sweep == 3 and s.trials == 3 * reg.sum() and 0 < s.accepted < s.trials
    ref = s.demag_field()
    scale = max(np.abs(x).max() for x in ref)
    for a in range(3):
        assert np.abs(b[a] - ref[a]).max() <= 1e-12 * scale


def test_parallel_frozen_field_matches_serial_exact_statistically():
    """Appendix B: the parallel checkerboard scheme with the field frozen during the iteration and without
    the self term gives no statistical difference from the serial algorithm with exact demag energy changes.  Small
    ellipse (24 x 12 cells, 15 mT along the long axis, 300 K), 6 seeds per scheme, means over the second half of 400
    iterations of the magnetisation along the field <m_x> (the paper's observable, Fig. 12) and of <|m|>; Welch statistic
    within 3 sigma.  The acceptance RATE is not such an observable: the serial scheme's self term (mu0 V/2) dM N(0) dM > 0
    (~0.04 kT per move here) makes it accept about 1.5 % fewer moves, which the test records."""
    def run(seed, serial):
        s, reg = _ellipse(24, 12, seed)
        act = reg > 0
        (s.run_serial_exact if serial else s.run)(200)
        a0, t0 = s.accepted, s.trials
        mx = ml = 0.0
        for _ in range(20):
            (s.run_serial_exact if serial else s.run)(10)
            mx += s.m[0][act].mean(); ml += np.sqrt(s.m[0] ** 2 + s.m[1] ** 2 + s.m[2] ** 2)[act].mean()
        return np.array([mx / 20, ml / 20, (s.accepted - a0) / (s.trials - t0)])
    P = np.array([run(100 + q, False) for q in range(6)])
    S = np.array([run(200 + q, True) for q in range(6)])
    for q, label in enumerate(("<m_x>", "<|m|>")):
        se = np.sqrt(P[:, q].var(ddof=1) / 6 + S[:, q].var(ddof=1) / 6)
        assert abs(P[:, q].mean() - S[:, q].mean()) <= 3.0 * se + 1e-6, (label, P[:, q].mean(), S[:, q].mean(), se)
    assert 0.0 < P[:, 2].mean() - S[:, 2].mean() < 0.03


# ------------------------------------------------------------------------------------------------ Appendix B at the paper's size (slow)
def _switching_run(args):
    """Worker (own process, one OpenMP thread): the 80 x 40 x 1 ellipse of PAPER.md:133 (400 x 200 x 5 nm, 5 nm cells), brought
    to remanence along -x at zero field, then H = 12 kA/m along +x; returns <m_x> over the non-empty cells
    after every `stride` iterations."""
    import os
    os.environ["OMP_NUM_THREADS"] = "1"
    seed, serial, n_it, stride = args
    s, reg = _ellipse(80, 40, seed, B=(0.0, 0.0, 0.0))
    act = reg > 0
    s.set_m(*(np.array([-0.8675, 0.0, 0.0])[:, None] * reg[None, :]))
    s.run(150)                                          # remanence (the parallel scheme on both arms: a common start)
    s.set_field(4e-7 * np.pi * 12e3, 0.0, 0.0)
    step = s.run_serial_exact if serial else s.run
    out = []
    for _ in range(n_it // stride):
        step(stride)
        out.append(s.m[0][act].mean())
    return np.array(out)


@pytest.mark.slow
def test_appendix_b_switching_at_the_papers_size():
    """SURVEY 8(f) row 2 / PAPER.md:218, Fig. 12, at the paper's shape and length: 80 x 40 x 1 ellipse (2516 magnetic cells), from
    the remanent state along -x with H = 12 kA/m applied along +x, the magnetisation along the field recorded over 10 000
    iterations, for the parallel frozen-field scheme (Eq. (14), one field per iteration) and the serial scheme with the exact
    demag energy change and a field update after every accepted move.  The paper averages 500 switching events per scheme;
    the serial oracle costs 0.07 s per iteration on one core, so this runs 8 events per scheme (about 12 minutes on 8 cores;
    MMC_APPB_ITERS shortens it).  Criterion, fixed before looking at the data of the run that DESIGN.md quotes:
      (a) the repo's usual one on ONE number per event, the run average of <m_x>: Welch |difference| <= 3 standard errors;
      (b) every recorded iteration count (each 250 iterations): Welch t statistic within the two-sided Student-t quantile of
          the 3-sigma level (p = 0.0027) divided by the number of checkpoints (Bonferroni), at the Welch-Satterthwaite degrees
          of freedom of 8 + 8 events.  (A first version of this test used an ad-hoc bar of 3.5 for (b) and failed it with 3.52
          at one of 30 checkpoints of a 1500-iteration run; a normal quantile is the wrong bar for 8 events per arm.)
    Run with `pytest --runslow -m slow -s`; DESIGN.md quotes the printed line of the last run."""
    import multiprocessing as mp
    import os
    from scipy import stats
    n_it = int(os.environ.get("MMC_APPB_ITERS", "10000")); stride = 250; n_ev = 8
    jobs = [(300 + q, True, n_it, stride) for q in range(n_ev)] + [(500 + q, False, n_it, stride) for q in range(n_ev)]
    with mp.get_context("spawn").Pool(min(8, os.cpu_count() or 1)) as pool:
        res = pool.map(_switching_run, jobs, chunksize=1)
    S = np.array(res[:n_ev]); P = np.array(res[n_ev:])
    n_chk = S.shape[1]

    def welch(a, b):
        va, vb = a.var(ddof=1) / a.size, b.var(ddof=1) / b.size
        se2 = va + vb + 1e-12
        dof = se2 ** 2 / (va ** 2 / (a.size - 1) + vb ** 2 / (b.size - 1) + 1e-300)
        return abs(a.mean() - b.mean()) / np.sqrt(se2), dof
    worst_ratio = 0.0; worst_t = 0.0
    for q in range(n_chk):
        t, dof = welch(S[:, q], P[:, q])
        bar = stats.t.ppf(1.0 - 0.5 * 0.0027 / n_chk, max(dof, 1.0))
        if t / bar > worst_ratio:
            worst_ratio, worst_t = t / bar, t
    za, _ = welch(S.mean(axis=1), P.mean(axis=1))
    switched = lambda X: int((X[:, -1] > 0).sum())
    print(f"Appendix B, {n_ev} events x {n_it} iterations per scheme: final <m_x> serial {S[:, -1].mean():+.4f} parallel {P[:, -1].mean():+.4f}; "
          f"switched (m_x > 0 at the end) serial {switched(S)}/{n_ev} parallel {switched(P)}/{n_ev}; run average serial {S.mean():+.4f} "
          f"parallel {P.mean():+.4f}, Welch z {za:.2f}; worst checkpoint t {worst_t:.2f} = {worst_ratio:.2f} of its Bonferroni bar ({n_chk} checkpoints)")
    assert S[:, 0].mean() < -0.5 and P[:, 0].mean() < -0.5          # both start near the remanent -x state
    assert za <= 3.0 and worst_ratio <= 1.0
