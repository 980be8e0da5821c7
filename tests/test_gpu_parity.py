"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on identical seeded
inputs and identical Philox streams.  Tolerances (north_star):
  stage 1  |dm_gpu - dm_oracle| <= 2e-6 |m|                       (trial vectors; trigonometry in fp32)
  stage 2  |term_gpu - term_oracle| <= 1e-5 * sum|terms| per cell, every term and the total dF, NO allowance: the five
           direction-dependent terms against the oracle evaluated at the kernel's dm, the longitudinal term against the
           oracle's own pass (both hold the length factor f exactly), the total against their sum
  margin   |margin_gpu - (oracle logs + that dF)| <= 1e-5 * sum|terms| + 2e-7 |ln u - 4 ln f| + 1e-6
  decisions identical except cells with |margin_oracle| < 1e-4 + 2e-6 * sum|terms|
  demag    |B_gpu - B_oracle| <= 2e-5 * max|B_oracle|
"""
import numpy as np
import pytest

import oracle as O
import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _gpu(wl):
    import paper_2106_05593_b200 as P
    s = P.MMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask)
    W.configure(s, wl, P.Material)
    return s


def _orc(wl, **kw):
    s = O.OracleMMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, store_fp32=True)
    W.configure(s, wl, O.Material)
    for k, v in kw.items():
        setattr(s, k, v)
    return s


def _np(ts):
    return [t.detach().cpu().numpy().astype(np.float64) for t in ts]


class _env:
    """Set an environment variable for the duration of a block (the library reads its A/B knobs when a context / plan is created)."""
    def __init__(self, key, val): self.key, self.val = key, val
    def __enter__(self):
        import os
        self.old = os.environ.get(self.key); os.environ[self.key] = self.val
    def __exit__(self, *a):
        import os
        if self.old is None: os.environ.pop(self.key, None)
        else: os.environ[self.key] = self.old


STATS = []          # (worst term error, worst total error, worst margin error) per checked pass, in units of their bars


@pytest.fixture(scope="module", autouse=True)
def _report_stats():
    """With MMC_TEST_STATS=<file> the worst stage-2 / margin errors of the module (in units of their bars) are written out."""
    yield
    import json, os
    if os.environ.get("MMC_TEST_STATS") and STATS:
        a = np.array(STATS)
        with open(os.environ["MMC_TEST_STATS"], "w") as f:
            json.dump({"passes": len(STATS), "worst_term_over_bar": a[:, 0].max(), "worst_total_over_bar": a[:, 1].max(),
                       "worst_margin_over_bar": a[:, 2].max(), "median_term_over_bar": float(np.median(a[:, 0]))}, f)


def check_pass(g, o, colour, wl, allow_flip_frac=2e-3):
    """One colour pass on both sides from the GPU's current state; returns number of near-margin flips."""
    m_before = _np(g.get_m())
    o.set_m(*m_before)
    ob = g.observables()
    o.sweep = int(ob["sweeps_done"]); o.cone_deg = float(ob["cone_deg"])
    if wl.demag:
        o.bd = [b.astype(np.float64) for b in _np(g.demag_field())]   # same frozen field on both sides (demag has its own test)
        o.demag_enabled = True
    d = g.debug_pass(colour)
    od = o.colour_pass(colour, dump=True)
    gdm = d["dm"].cpu().numpy().astype(np.float64); gt = d["terms"].cpu().numpy().astype(np.float64)
    gmar = d["margin"].cpu().numpy().astype(np.float64); gacc = d["accepted"].cpu().numpy()
    act = ~np.isnan(od["margin"])
    assert np.array_equal(act, gacc != 255), "set of cells that received a trial differs"
    assert act.sum() > 0 or wl.n_active == 0
    L = np.sqrt(m_before[0] ** 2 + m_before[1] ** 2 + m_before[2] ** 2)
    # stage 1
    err1 = np.abs(gdm[act] - od["dm"][act]).max(axis=1)
    assert np.all(err1 <= 2e-6 * L[act]), f"stage 1: max {np.max(err1 / L[act]):.3e}"
    # stage 2: oracle energy arithmetic on the GPU's trial vectors, from the pre-pass state
    o2 = _orc(wl); o2.set_m(*m_before); o2.sweep = o.sweep; o2.cone_deg = o.cone_deg
    if wl.demag:
        o2.bd = o.bd; o2.demag_enabled = True
    ot = o2.colour_terms_given_dm(colour, np.where(np.isnan(gdm), 0.0, gdm))
    own = od["terms"][act]                            # the oracle's OWN pass: fp64 dm, |m'| = f |m| exactly (O3)
    # The bar of north_star / G15, no allowance anywhere: 1e-5 * sum |terms| per cell, for
    #   (a) the five direction-dependent terms (ex, an, zee, dmi, demag) against the oracle evaluated at the kernel's dm;
    #   (b) the longitudinal term against the oracle's own pass: it depends on the move only through the length factor
    #       f = 1 + sigma (2u - 1), which both sides hold exactly, so both describe the same ideal move;
    #   (c) the total dF against (a) + (b): the oracle's dF/kBT of the kernel's trial move with |m'| = f |m|.
    hyb = ot[act].copy(); hyb[:, 5] = own[:, 5]
    scale = np.abs(hyb).sum(axis=1)
    err2 = np.abs(gt[act] - hyb)
    bar = 1e-5 * scale + 1e-30
    worst = err2 / bar[:, None]
    assert np.all(err2 <= bar[:, None]), f"stage 2: worst {worst.max():.3f} x the 1e-5 bar (term {np.argmax(worst.max(axis=0))})"
    tot = np.abs(gt[act].sum(axis=1) - hyb.sum(axis=1))
    assert np.all(tot <= bar), f"stage 2 total: worst {np.max(tot / bar):.3f} x the 1e-5 bar"
    # Diagnostic (2'), with an allowance, of how well the kernel's STORED trial vector honours |m + dm| = f |m|: the oracle
    # forms dl2 = dm.(2m+dm) from the kernel's fp32 dm, in which the rotation part cancels, so that dl2 carries the fp32
    # noise of dm: half an ulp per stored component (2^-24 |dm| sqrt 3) plus the ~1 ulp (2^-23) normalisation error of the
    # kernel's unit vectors n, t1, t2, which scales |m + dm| by up to 4 ulp.  d(long)/d(dl2) = c4 (2 l2 + 2 dl2) + c2.
    # (DESIGN.md section 5 row 2' lists both summands; the kernel itself takes dl2 = l2 s (2 + s), reading P(i').)
    o2._setup()
    c4 = o2.coef["c4"][act]; c2 = o2.coef["c2"][act]
    gd = np.where(np.isnan(gdm), 0.0, gdm)[act]
    l2 = L[act] ** 2
    dl2 = sum(gd[:, a] * (2 * m_before[a][act] + gd[:, a]) for a in range(3))
    ddl2 = 2.0 * L[act] * (np.linalg.norm(gd, axis=1) * 2.0 ** -24 * np.sqrt(3.0) + L[act] * 4 * 2.0 ** -23)
    allow = np.abs(c4 * (2.0 * l2 + 2.0 * dl2) + c2) * ddl2
    assert np.all(np.abs(gt[act][:, 5] - ot[act][:, 5]) <= bar + allow), "stored trial vector: |m + dm| deviates from f |m| by more than 4 ulp"
    # decisions
    omar = od["margin"][act]
    flips = (gacc[act] != od["accepted"][act])
    window = 1e-4 + 2e-6 * np.abs(own).sum(axis=1)
    assert np.all(np.abs(omar[flips]) < window[flips]), "decision differs outside the margin window"
    assert flips.sum() <= max(1, allow_flip_frac * act.sum())
    # margin = ln u - 4 ln f + dF: the oracle's logarithms (its margin minus its dF) plus the hybrid dF above; the kernel's
    # two MUFU lg2 carry 2^-22 relative each (|ln u| <= 16.7), the fp32 sum half an ulp of the largest partial sum
    olog = omar - own.sum(axis=1)
    mbar = bar + 2e-7 * np.abs(olog) + 1e-6
    merr = np.abs(gmar[act] - (olog + hyb.sum(axis=1)))
    assert np.all(merr <= mbar), f"margin: worst {np.max(merr / mbar):.3f} x its bar"
    STATS.append((float(worst.max()), float(np.max(tot / bar)), float(np.max(merr / mbar))))
    # state after the pass: identical where decisions agree (fp32 storage on both sides)
    m_after = _np(g.get_m())
    same = np.ones(wl.N, bool); idx = np.flatnonzero(act)[flips]; same[idx] = False
    for a in range(3):
        assert np.allclose(m_after[a][same], o.m[a][same], rtol=0, atol=2.5e-6 * max(1e-3, L.max()))
        assert np.array_equal(m_after[a][~act], m_before[a][~act])
    return int(flips.sum()), int(act.sum()), int(gacc[act].sum())


def _small(cfg, **kw):
    return W.make(cfg, **kw)


def _with_pbc(wl, mask):
    wl.pbc_mask = mask                                # exchange / DMI wrap; the demag convolution stays open-boundary
    return wl


def _with_k2(wl, K2):
    for r in wl.regions:
        if r["Ms0"] > 0:
            r["K2"] = K2                              # 4th-order uniaxial term of Eq. (11)
    return wl


CASES = {
    "cfg1_32x32": lambda: W.cfg1(),
    "cfg1_paper_regime": lambda: W.cfg1(paper_regime=True),
    "cfg1_ragged_40x24": lambda: W.cfg1(nx=40, ny=24, paper_regime=True),      # nx % 8 == 0 but not a power of two
    "cfg1_ragged_periodic_12x6": lambda: W.cfg1(nx=12, ny=6, paper_regime=True),  # padded compact rows + periodic wrap
    "cfg2_64x48": lambda: W.cfg2(nx=64, ny=48),
    "cfg2_ragged_37x19": lambda: W.cfg2(nx=37, ny=19),                         # odd sizes, open boundaries
    "cfg3_64x64_200K": lambda: W.cfg3(nx=64, ny=64, T=200.0),
    "cfg3_64x64_700K_Tc": lambda: W.cfg3(nx=64, ny=64, T=700.0),               # T == Tc exactly (G10)
    "cfg3_48x40_800K": lambda: W.cfg3(nx=48, ny=40, T=800.0),
    "cfg4_48x40x4": lambda: W.cfg4(nx=48, ny=40, nz=4),
    "cfg4_30x21x3": lambda: W.cfg4(nx=30, ny=21, nz=3),
    "cfg5_160x150": lambda: W.cfg5(nx=160, ny=150),
    # cubic anisotropy (Eq. (12), K1c + K2c, random cubic axes per grain), periodic in the plane, phase-separated grains
    "fe_film_cubic_48x40x3": lambda: W.fe_film(nx=48, ny=40, nz=3),
    "fe_film_cubic_36x22x10": lambda: W.fe_film(nx=36, ny=22, nz=10),
    # K1 + K2 of Eq. (11): uniform film (kernel arguments) and granular film (class tables, tilted axes, T > Tc in the hot spot)
    "cfg1_k2_32x32": lambda: _with_k2(W.cfg1(paper_regime=True), -1.5e5),
    "cfg4_k2_30x21x3": lambda: _with_k2(W.cfg4(nx=30, ny=21, nz=3), 4e5),
    # periodic directions not covered by the recipes: z wrap (also with the two z neighbours being the same cell), wrap in all
    # three directions on per-cell classes, y wrap on odd nx (padded compact rows), and the shortest periodic lengths
    "cfg4_periodic_xyz_16x12x4": lambda: _with_pbc(W.cfg4(nx=16, ny=12, nz=4), 0b111),
    "cfg4_periodic_z_15x9x2": lambda: _with_pbc(W.cfg4(nx=15, ny=9, nz=2), 0b100),
    "cfg2_periodic_y_37x20": lambda: _with_pbc(W.cfg2(nx=37, ny=20), 0b010),
    "cfg3_periodic_dmi_2x2": lambda: W.cfg3(nx=2, ny=2, T=200.0),
    "cfg1_periodic_2x6": lambda: W.cfg1(nx=2, ny=6, paper_regime=True),
    # periodic in x with an ODD compact row length (nx/2 = 5, 7): the wrap neighbour of a row's last cell does not pair up, so these
    # meshes always take the one-cell-per-thread kernel (launch_variant, "pairable")
    "cfg1_periodic_odd_rows_10x6": lambda: W.cfg1(nx=10, ny=6, paper_regime=True),
    "cfg3_periodic_dmi_odd_rows_14x10": lambda: W.cfg3(nx=14, ny=10, T=200.0),
}


@pytest.mark.parametrize("name", list(CASES))
def test_colour_pass_parity(name):
    wl = CASES[name]()
    if name.startswith("cfg3") and "Tc" not in name and "800K" not in name:
        wl.cone_deg = 12.0
    g, o = _gpu(wl), _orc(wl)
    flips = trials = accepted = 0
    for sweep in range(2):
        for colour in (0, 1):
            f, t, a = check_pass(g, o, colour, wl)
            flips += f; trials += t; accepted += a
        g.set_sweep_counter(sweep + 1)
    assert trials == 2 * wl.n_active
    ob = g.observables()
    assert ob["trials"] == trials and ob["accepted"] == accepted
    g.close()


def _check_iteration(wl, g, o, label):
    """One whole iteration of the production kernels against the oracle's replay, every differing cell explained
    (tests/parity_util.py); returns the classification."""
    from parity_util import explain_iteration
    g.sweep(1)
    r = explain_iteration(wl, o, _np(g.get_m()))
    assert r["untouched_ok"], f"{label}: a cell without a trial changed"
    assert r["neither"] == 0, f"{label}: {r['neither']} cells hold neither the accepted nor the rejected candidate"
    assert r["unexplained"] == 0, f"{label}: {r['unexplained']} of {r['flips']} decision flips are not explained by the oracle's margins"
    assert r["flips"] <= max(2, 2e-3 * wl.n_active), f"{label}: {r['flips']} flips"
    ob = g.observables()
    assert ob["trials"] == r["active"] == wl.n_active
    assert abs(int(ob["accepted"]) - r["oracle_accepted"]) <= r["flips"]
    return r


@pytest.mark.parametrize("name", ["cfg1_paper_regime", "cfg2_ragged_37x19", "cfg3_64x64_200K", "cfg4_30x21x3", "cfg5_160x150",
                                  "fe_film_cubic_48x40x3", "cfg4_k2_30x21x3", "cfg4_periodic_xyz_16x12x4", "cfg4_periodic_z_15x9x2",
                                  "cfg2_periodic_y_37x20", "cfg3_periodic_dmi_2x2", "cfg1_periodic_2x6", "cfg1_periodic_odd_rows_10x6",
                                  "cfg3_periodic_dmi_odd_rows_14x10"])
@pytest.mark.parametrize("cells", ["two_cells_per_thread", "one_cell_per_thread"])
def test_sweep_matches_replayed_oracle(name, cells):
    """mmc_sweep(n) (demag -> red -> black -> counter++) against the oracle replaying the same iteration, each side with its
    own demag field.  Every active cell must hold the oracle's accepted or rejected candidate, and every cell whose decision
    differs must be a near-margin decision by the oracle's own margin (or a black neighbour of a red one).  With both pass
    kernels: grids of fewer CTAs than SMs -- every mesh here -- take the one-cell-per-thread kernel by default, the paper-sized
    meshes the two-cell kernel (MMC_PASS1_BELOW, include/mmc.h)."""
    wl = CASES[name]()
    wl.adaptive_cone = False
    with _env("MMC_PASS1_BELOW", "0" if cells == "two_cells_per_thread" else "1000000"):
        g = _gpu(wl)
    o = _orc(wl)
    _check_iteration(wl, g, o, name)
    assert g.observables()["sweeps_done"] == 1
    g.close()


@pytest.mark.parametrize("name", ["cfg2_64x48", "cfg2_ragged_37x19", "cfg3_64x64_200K", "cfg4_48x40x4", "cfg4_30x21x3", "cfg5_160x150",
                                  "fe_film_cubic_48x40x3", "cfg4_periodic_xyz_16x12x4", "cfg2_periodic_y_37x20", "cfg1_ragged_40x24"])
def test_pass_kernels_with_one_and_two_cells_per_thread_agree_bitwise(name):
    """Same cell arithmetic in both kernels: states, counters, cone and energies agree bit for bit after 25 iterations; the
    running means to their fixed-point quantum (the two-cell kernel rounds the sum of a thread's pair, the other every cell)."""
    wl = CASES[name]()
    wl.adaptive_cone = True
    with _env("MMC_PASS1_BELOW", "0"):
        a = _gpu(wl)
    with _env("MMC_PASS1_BELOW", "1000000"):
        b = _gpu(wl)
    a.sweep(25); b.sweep(25)
    ma, mb = a.get_m(), b.get_m()
    assert all(bool((ma[q] == mb[q]).all()) for q in range(3))
    oa, ob = a.observables(), b.observables()
    for k in ("accepted", "trials", "sweeps_done", "cone_deg", "run_sweeps", "E_ex", "E_an", "E_demag", "E_long"):
        assert oa[k] == ob[k], k
    assert abs(oa["run_mean_len"] - ob["run_mean_len"]) < 2.0 ** -22 and np.abs(oa["run_mean_m"] - ob["run_mean_m"]).max() < 2.0 ** -22
    a.close(); b.close()


def test_cfg1_as_written_1000_sweeps_in_lockstep():
    """BASELINE.json config 1 exactly as written (32x32x1, PBC, sigma = 0.05, cone 30 deg fixed, 1000 sweeps, no demag):
    the CUDA path (the single-launch small-mesh kernel, one iteration per call) against the oracle in lockstep.  After
    EVERY iteration each cell holds the oracle's accepted or rejected candidate and every differing decision is explained by
    the oracle's margin; after an explained flip the oracle continues from the CUDA path's state, so the comparison stays
    cell-exact over all 1000 iterations instead of decorrelating.  Counters agree up to the flips; the final observables
    agree to fp32 storage."""
    from parity_util import explain_iteration
    wl = W.cfg1()
    g, o = _gpu(wl), _orc(wl)
    flips = oacc = 0
    for it in range(1000):
        g.sweep(1)
        mg = _np(g.get_m())
        r = explain_iteration(wl, o, mg)
        assert r["neither"] == 0 and r["unexplained"] == 0 and r["untouched_ok"], (it, r)
        flips += r["flips"]; oacc += r["oracle_accepted"]
        if r["flips"]:
            o.set_m(*mg)
    ob, oo = g.observables(), o.observables()
    assert ob["sweeps_done"] == 1000 and ob["trials"] == 1000 * wl.N
    assert abs(int(ob["accepted"]) - oacc) <= flips <= 20, (ob["accepted"], oacc, flips)
    assert 0.002 < ob["accepted"] / ob["trials"] < 0.05           # sigma = 0.05 >> the width of the length distribution: ~1 %
    assert np.allclose(ob["mean_m"], oo["mean_m"], atol=1e-6) and ob["mean_len"] == pytest.approx(oo["mean_len"], rel=1e-6)
    for k in ("E_ex", "E_an", "E_long"):
        assert ob[k] == pytest.approx(oo[k], rel=2e-5), k
    g.close()


def _stirred(wl, seed):
    """The workload with a random initial state (unit vectors times the recipe's lengths) and a wide cone: the red pass then
    changes the demag field by several percent, so a second field update before the black pass changes many decisions."""
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(3, wl.N)); v /= np.linalg.norm(v, axis=0)
    L = np.sqrt(sum(wl.m0[a].astype(np.float64) ** 2 for a in range(3)))
    wl.m0 = np.stack([(L * v[a]).astype(np.float32) for a in range(3)])
    wl.cone_deg = 40.0; wl.adaptive_cone = False
    return wl


@pytest.mark.parametrize("exchange", [True, False], ids=["with_exchange", "demag_only"])
@pytest.mark.parametrize("name", ["cfg2_64x48", "cfg2_ragged_37x19", "cfg4_48x40x4", "cfg4_30x21x3", "cfg5_160x150"])
def test_two_demag_updates_per_iteration(name, exchange):
    """"the demagnetizing field can be updated before each red and black parallel passes" (SURVEY 8(f) row 2,
    reading G12): mmc_set_demag(ctx, 1, 2) against OracleMMC.set_demag(True, 2), one whole iteration from a stirred state.
    With the recipe's exchange the decisions are dominated by |dF_ex| and only a few black cells notice the
    second update; in the demag_only variant (A0 = 0, K1 = 0: the field is the only direction-dependent term) the oracle
    alone shows that one and two updates decide differently in many black cells, and the CUDA path must side with two
    updates in all of them (up to explained near-margin flips)."""
    wl = _stirred(CASES[name](), 77)
    if not exchange:
        for r in wl.regions:
            r["A0"] = 0.0; r["K1"] = 0.0
    g, o2, o1 = _gpu(wl), _orc(wl), _orc(wl)
    g.set_demag(True, 2); o2.set_demag(True, 2); o1.set_demag(True, 1)
    r = _check_iteration(wl, g, o2, name + " (2 updates)")
    o1.run(1)
    differ = np.zeros(wl.N, bool)
    for a in range(3):
        differ |= np.abs(o1.m[a] - o2.m[a]) > 2e-6
    if not exchange:
        assert differ.sum() >= 3, f"only {differ.sum()} cells distinguish one from two field updates"   # oracle alone: 113, 18, 8, 3, 170
    mg = _np(g.get_m())
    side2 = np.ones(wl.N, bool)
    for a in range(3):
        side2 &= np.abs(mg[a] - o2.m[a]) <= 2e-6
    assert (differ & ~side2).sum() <= r["flips"], "black cells follow the one-update field"
    # and back: one update per iteration again gives the one-update result
    h = _gpu(wl); h.set_demag(True, 2); h.set_demag(True, 1)
    _check_iteration(wl, h, _orc(wl), name + " (1 update)")
    g.close(); h.close()


@pytest.mark.parametrize("shape,d", [((64, 48, 1), (5e-9, 5e-9, 5e-9)), ((37, 19, 1), (5e-9, 5e-9, 10e-9)),
                                     ((48, 40, 4), (3e-9, 3e-9, 3e-9)), ((30, 21, 3), (2e-9, 3e-9, 4e-9)),
                                     ((128, 96, 1), (5e-9, 5e-9, 10e-9)),
                                     # column transforms of length 2^8 .. 2^12 (register-resident kernels), with the
                                     # padding exactly half (pruned variant) and ragged, one and several layers
                                     ((128, 128, 1), (5e-9, 5e-9, 5e-9)), ((100, 200, 1), (5e-9, 4e-9, 3e-9)),
                                     ((64, 256, 2), (3e-9, 3e-9, 3e-9)), ((72, 512, 1), (2e-9, 2e-9, 2e-9)),
                                     ((40, 600, 1), (5e-9, 5e-9, 10e-9)), ((48, 1024, 2), (3e-9, 3e-9, 3e-9)),
                                     ((20, 700, 3), (3e-9, 3e-9, 3e-9)),
                                     ((32, 2048, 1), (5e-9, 5e-9, 10e-9)), ((36, 1100, 1), (5e-9, 5e-9, 5e-9)),
                                     # row transforms of length 2^8 .. 2^11 (register-resident kernels): 1, 2, 3, 4, 5 layers
                                     # (padded z length 1, 4, 8, 8, 16), ragged row tiles, odd nx
                                     ((200, 40, 1), (5e-9, 5e-9, 5e-9)), ((256, 22, 4), (3e-9, 3e-9, 3e-9)),
                                     ((301, 18, 3), (2e-9, 3e-9, 4e-9)), ((512, 16, 2), (3e-9, 3e-9, 3e-9)),
                                     ((1024, 10, 1), (5e-9, 5e-9, 10e-9)), ((700, 9, 4), (3e-9, 3e-9, 3e-9)),
                                     ((520, 6, 5), (3e-9, 3e-9, 3e-9)), ((2048, 7, 1), (5e-9, 5e-9, 10e-9)),
                                     ((1500, 5, 2), (3e-9, 3e-9, 3e-9)),
                                     # register-resident rows AND columns kernels: one layer (planar columns kernel), 2 - 4 layers
                                     # (layer-pair columns kernel, no z transform), 10 and 16 layers (z-DFT of length 2 nz - 1
                                     # in the columns kernel's loader + the inverse z pass); ragged chunks
                                     ((256, 256, 1), (5e-9, 5e-9, 5e-9)), ((512, 128, 4), (3e-9, 3e-9, 3e-9)),
                                     ((200, 70, 1), (5e-9, 5e-9, 5e-9)), ((256, 66, 4), (3e-9, 3e-9, 3e-9)),
                                     ((301, 67, 3), (2e-9, 3e-9, 4e-9)), ((512, 72, 2), (3e-9, 3e-9, 3e-9)),
                                     ((1024, 65, 1), (5e-9, 5e-9, 10e-9)), ((700, 69, 4), (3e-9, 3e-9, 3e-9)),
                                     ((2048, 66, 1), (5e-9, 5e-9, 10e-9)), ((1500, 65, 2), (3e-9, 3e-9, 3e-9)),
                                     ((130, 300, 3), (3e-9, 3e-9, 3e-9)), ((132, 70, 10), (2e-9, 2e-9, 2e-9)),
                                     ((256, 65, 16), (2e-9, 2e-9, 2e-9)),
                                     # register-resident path with every other layer count up to 16 (z-DFT lengths 9 .. 29)
                                     ((130, 65, 5), (3e-9, 3e-9, 3e-9)), ((130, 70, 6), (3e-9, 3e-9, 2e-9)), ((140, 65, 7), (3e-9, 3e-9, 3e-9)),
                                     ((130, 66, 8), (2e-9, 3e-9, 3e-9)), ((130, 65, 9), (3e-9, 3e-9, 3e-9)), ((130, 65, 11), (3e-9, 3e-9, 3e-9)),
                                     ((129, 65, 12), (3e-9, 3e-9, 3e-9)), ((130, 65, 13), (3e-9, 3e-9, 4e-9)), ((130, 67, 14), (3e-9, 3e-9, 3e-9)),
                                     ((130, 65, 15), (3e-9, 3e-9, 3e-9)),
                                     # generic shared-memory kernels (nx <= 128) with 9 .. 16 layers: padded z length 32
                                     ((64, 48, 10), (2e-9, 2e-9, 2e-9)), ((40, 24, 16), (3e-9, 2e-9, 2e-9)), ((96, 20, 9), (2e-9, 2e-9, 4e-9))])
def test_demag_field_parity(shape, d):
    """Eq. (14): GPU fp32 FFT convolution vs the oracle's fp64 one (itself pinned to the direct sum)."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(N)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (v * rng.uniform(0.3, 1.0, N)).astype(np.float32)
    reg = (rng.uniform(size=N) > 0.2).astype(np.int32)
    m0[:, reg == 0] = 0
    g = P.MMC(nx, ny, nz, *d, 0)
    g.set_material([P.Material(), P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)], reg)
    g.set_temperature(300.0); g.set_m(*m0)
    bg = _np(g.demag_field())
    conv = O.DemagFFT(nx, ny, nz, *d)
    M = [(8.6e5 * reg * m0[a].astype(np.float64)).reshape(nz, ny, nx) for a in range(3)]
    bo = [b.ravel() for b in conv.field(*M)]
    scale = max(np.abs(b).max() for b in bo)
    for a in range(3):
        assert np.abs(bg[a] - bo[a]).max() <= 2e-5 * scale
    g.close()


@pytest.mark.parametrize("shape,d", [((1, 1, 1), (5e-9, 5e-9, 5e-9)), ((1, 1, 5), (5e-9, 4e-9, 3e-9)), ((7, 1, 1), (2e-9, 3e-9, 4e-9)),
                                     ((1, 9, 1), (2e-9, 3e-9, 4e-9)), ((2, 2, 2), (3e-9, 3e-9, 3e-9)), ((1, 5, 3), (3e-9, 3e-9, 5e-9)),
                                     ((2, 1, 16), (3e-9, 3e-9, 3e-9)),
                                     # beyond the register-resident lengths: padded nx 8192 (generic rows kernels, with generic and
                                     # with register-resident columns), padded ny 8192 (generic columns kernel, 209 KB of shared memory)
                                     ((2100, 6, 1), (5e-9, 5e-9, 10e-9)), ((2100, 130, 2), (3e-9, 3e-9, 3e-9)), ((12, 2100, 1), (5e-9, 5e-9, 5e-9))])
def test_demag_field_parity_degenerate_and_oversize_meshes(shape, d):
    """Eq. (14) on meshes with directions of length 1 or 2 (padded lengths 1, 2, 4: self-term and nearest offsets only) and on
    meshes longer than the register-resident transforms serve; every cell magnetic."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(1000 + N)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (v * rng.uniform(0.3, 1.0, N)).astype(np.float32)
    g = P.MMC(nx, ny, nz, *d, 0)
    g.set_material([P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)])
    g.set_temperature(300.0); g.set_m(*m0)
    bg = _np(g.demag_field())
    conv = O.DemagFFT(nx, ny, nz, *d)
    M = [(8.6e5 * m0[a].astype(np.float64)).reshape(nz, ny, nx) for a in range(3)]
    bo = [b.ravel() for b in conv.field(*M)]
    scale = max(np.abs(b).max() for b in bo)
    assert scale > 0.1                                                # tesla: a saturated cell's own field
    for a in range(3):
        assert np.abs(bg[a] - bo[a]).max() <= 2e-5 * scale
    g.close()


@pytest.mark.parametrize("shape", [(256, 256, 1), (100, 200, 1), (200, 70, 1), (1024, 65, 1)])
def test_split_and_unsplit_planar_columns_kernel_agree_bitwise(shape):
    """One-layer meshes: the in-plane pair and the z component of the columns kernel in one CTA (MMC_COLS_SPLIT=0) or in two (=1; the
    default below two CTAs per SM): the same arithmetic per element, so the same bits."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(N + 11)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (v * rng.uniform(0.3, 1.0, N)).astype(np.float32)
    out = []
    for split in ("0", "1"):
        with _env("MMC_COLS_SPLIT", split):
            g = P.MMC(nx, ny, nz, 5e-9, 5e-9, 5e-9, 0)
            g.set_material([P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)]); g.set_temperature(300.0); g.set_m(*m0)
            out.append([b.clone() for b in g.demag_field()])
            g.close()
    assert all(torch.equal(out[0][a], out[1][a]) for a in range(3))
    assert float(out[0][2].abs().max()) > 0.1


def test_demag_more_than_16_layers_is_a_clean_error():
    import paper_2106_05593_b200 as P
    g = P.MMC(4, 4, 17, 3e-9, 3e-9, 3e-9, 0)
    g.set_material([P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)]); g.set_temperature(300.0)
    g.set_m(np.zeros(272), np.zeros(272), np.full(272, 0.9))
    with pytest.raises(P.MMCError) as e:
        g.demag_field()
    assert e.value.code == -5 and "16 layers" in str(e.value)
    g.sweep(2)                                                        # the context still works without demag
    assert g.observables()["trials"] == 2 * 272
    g.close()


@pytest.mark.parametrize("shape,d", [((256, 256, 1), (5e-9, 5e-9, 5e-9)), ((301, 67, 3), (2e-9, 3e-9, 4e-9)), ((512, 72, 2), (3e-9, 3e-9, 3e-9)),
                                     ((256, 66, 4), (3e-9, 3e-9, 3e-9)), ((200, 300, 5), (3e-9, 3e-9, 3e-9)), ((132, 70, 10), (2e-9, 2e-9, 2e-9)),
                                     ((256, 65, 16), (2e-9, 2e-9, 2e-9))])
def test_generic_demag_kernels_on_meshes_the_fast_path_serves(shape, d):
    """MMC_DEMAG_GENERIC=1: the any-length shared-memory kernels (rows with the z transform of padded length 1 .. 32 in registers,
    columns per (kx, kz)) on shapes that normally take the register-resident kernels: same bar against the oracle."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(N + 3)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (v * rng.uniform(0.3, 1.0, N)).astype(np.float32)
    reg = (rng.uniform(size=N) > 0.2).astype(np.int32)
    m0[:, reg == 0] = 0
    with _env("MMC_DEMAG_GENERIC", "1"):
        g = P.MMC(nx, ny, nz, *d, 0)
        g.set_material([P.Material(), P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)], reg)
        g.set_temperature(300.0); g.set_m(*m0)
        bg = _np(g.demag_field())
    conv = O.DemagFFT(nx, ny, nz, *d)
    M = [(8.6e5 * reg * m0[a].astype(np.float64)).reshape(nz, ny, nx) for a in range(3)]
    bo = [b.ravel() for b in conv.field(*M)]
    scale = max(np.abs(b).max() for b in bo)
    for a in range(3):
        assert np.abs(bg[a] - bo[a]).max() <= 2e-5 * scale
    g.close()


@pytest.mark.parametrize("shape,d", [((64, 256, 2), (3e-9, 3e-9, 3e-9)), ((48, 1024, 2), (3e-9, 3e-9, 3e-9)), ((130, 300, 3), (3e-9, 3e-9, 3e-9)),
                                     ((512, 128, 4), (3e-9, 3e-9, 3e-9)), ((256, 66, 4), (3e-9, 3e-9, 3e-9)), ((301, 67, 3), (2e-9, 3e-9, 4e-9)),
                                     ((700, 69, 4), (3e-9, 3e-9, 3e-9)), ((200, 2048, 2), (3e-9, 3e-9, 3e-9))])
def test_layer_pair_columns_kernel_parity(shape, d):
    """The layer-pair variant of the columns kernel (MMC_LP=1: no z transform, layers combined per frequency with the 2-D tensor
    spectra of the layer offsets; Eq. (14) written out in z) against the oracle's fp64 convolution: same bar as the default path."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(N + 7)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (v * rng.uniform(0.3, 1.0, N)).astype(np.float32)
    reg = (rng.uniform(size=N) > 0.2).astype(np.int32)
    m0[:, reg == 0] = 0
    with _env("MMC_LP", "1"):
        g = P.MMC(nx, ny, nz, *d, 0)
        g.set_material([P.Material(), P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)], reg)
        g.set_temperature(300.0); g.set_m(*m0)
        bg = _np(g.demag_field())
        again = _np(g.demag_field())
    conv = O.DemagFFT(nx, ny, nz, *d)
    M = [(8.6e5 * reg * m0[a].astype(np.float64)).reshape(nz, ny, nx) for a in range(3)]
    bo = [b.ravel() for b in conv.field(*M)]
    scale = max(np.abs(b).max() for b in bo)
    for a in range(3):
        assert np.abs(bg[a] - bo[a]).max() <= 2e-5 * scale
        assert np.array_equal(bg[a], again[a])                       # deterministic (mbarrier / bulk-copy pipeline, shared-memory exchange)
    g.close()


@pytest.mark.parametrize("shape,d", [((130, 1024, 2), (3e-9, 3e-9, 3e-9)), ((130, 700, 3), (3e-9, 3e-9, 3e-9)), ((130, 512, 2), (3e-9, 3e-9, 3e-9)),
                                     ((130, 300, 3), (2e-9, 3e-9, 4e-9)), ((130, 2048, 2), (3e-9, 3e-9, 3e-9)), ((130, 1100, 2), (3e-9, 3e-9, 3e-9)),
                                     ((256, 1024, 4), (3e-9, 3e-9, 3e-9)), ((130, 1024, 7), (3e-9, 3e-9, 3e-9))])
def test_eight_point_columns_kernel_parity(shape, d):
    """The columns kernel with eight points per thread (MMC_COLS8=1, fft_reg8.cuh: 8 x 8 x 8 x T3 transforms of length 2^10 .. 2^12,
    padding exactly half and ragged, 2 - 7 layers) and the default kernel (16 points per thread) on the same mesh, both against the
    oracle's fp64 convolution at the default path's bar."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(N + 13)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (v * rng.uniform(0.3, 1.0, N)).astype(np.float32)
    reg = (rng.uniform(size=N) > 0.2).astype(np.int32)
    m0[:, reg == 0] = 0
    out = {}
    for k in ("0", "1"):
        with _env("MMC_COLS8", k):
            g = P.MMC(nx, ny, nz, *d, 0)
            g.set_material([P.Material(), P.Material(Ms0=8.6e5, A0=1.3e-11, Tc=870.0)], reg)
            g.set_temperature(300.0); g.set_m(*m0)
            out[k] = _np(g.demag_field())
            if k == "1":
                again = _np(g.demag_field())
            g.close()
    conv = O.DemagFFT(nx, ny, nz, *d)
    M = [(8.6e5 * reg * m0[a].astype(np.float64)).reshape(nz, ny, nx) for a in range(3)]
    bo = [b.ravel() for b in conv.field(*M)]
    scale = max(np.abs(b).max() for b in bo)
    for a in range(3):
        assert np.abs(out["0"][a] - bo[a]).max() <= 2e-5 * scale
        assert np.abs(out["1"][a] - bo[a]).max() <= 2e-5 * scale
        assert np.array_equal(out["1"][a], again[a])
    assert any(not np.array_equal(out["0"][a], out["1"][a]) for a in range(3))      # a different transform did run


@pytest.mark.parametrize("name", ["cfg2_64x48", "cfg4_48x40x4", "cfg4_30x21x3", "cfg5_160x150"])
def test_tma_staged_pass_is_bitwise_the_default_pass(name):
    """The TMA-staged colour pass (MMC_TMA=1: cp.async.bulk.tensor boxes into a ring of shared-memory stages, warp-specialised)
    against the default pass (per-thread loads through L1): same cell arithmetic (update_pair), same integer reductions, so
    states, counters and running sums must agree bit for bit.  Meshes here are stretched in x and y so that the staged variant has
    the 296 tiles it asks for (smaller meshes fall back to the default kernel, which the test would then compare with itself)."""
    import paper_2106_05593_b200 as P
    base = CASES[name]()
    big = {"cfg2": lambda: W.cfg2(nx=1300, ny=500), "cfg4": lambda: W.cfg4(nx=1290, ny=190, nz=base.nz), "cfg5": lambda: W.cfg5(nx=1300, ny=500)}[name[:4]]
    out = []
    for tma in ("1", "0"):
        wl = big(); wl.adaptive_cone = False
        if name.startswith("cfg5"):
            wl.region_of_cell = np.ones(wl.N, np.int32); wl.m0 = np.tile(np.array([[0.5], [0.5], [0.2]], np.float32), (1, wl.N))   # mostly magnetic: staged
        with _env("MMC_TMA", tma):
            g = _gpu(wl)
            g.sweep(3)
            out.append(([x.clone() for x in g.get_m()], g.observables()))
            g.close()
    (ma, oa), (mb, ob) = out
    assert all(bool((ma[q] == mb[q]).all()) for q in range(3))
    for k in ("accepted", "trials", "run_mean_len", "E_ex", "E_demag"):
        assert oa[k] == ob[k], k
    assert np.array_equal(oa["run_mean_m"], ob["run_mean_m"]) and oa["trials"] == 3 * wl.n_active


@pytest.mark.parametrize("name", ["cfg1_32x32", "cfg2_ragged_37x19", "cfg3_64x64_200K", "cfg3_48x40_800K", "cfg4_30x21x3", "cfg5_160x150",
                                  "fe_film_cubic_48x40x3", "cfg1_k2_32x32", "cfg4_k2_30x21x3"])
def test_observables_parity(name):
    wl = CASES[name]()
    g, o = _gpu(wl), _orc(wl)
    og, oo = g.observables(), o.observables()
    assert np.allclose(og["mean_m"], oo["mean_m"], atol=1e-6)
    assert og["mean_len"] == pytest.approx(oo["mean_len"], rel=1e-6)
    tot = sum(abs(oo[k]) for k in ("E_ex", "E_an", "E_zee", "E_dmi", "E_demag", "E_long"))
    for k in ("E_ex", "E_an", "E_zee", "E_dmi", "E_demag", "E_long"):
        assert og[k] == pytest.approx(oo[k], rel=2e-5, abs=2e-6 * tot), k
    g.close()


def test_running_means_and_counters():
    wl = W.cfg1(paper_regime=True)
    g = _gpu(wl)
    g.reset_averages()
    means = []
    for _ in range(5):
        g.sweep(1)
        means.append(g.observables()["mean_m"])
    ob = g.observables()
    assert ob["run_sweeps"] == 5
    assert np.allclose(ob["run_mean_m"], np.mean(means, axis=0), atol=2e-6)
    assert ob["trials"] == 5 * wl.N and 0 < ob["accepted"] < ob["trials"]
    g.reset_counters()
    assert g.observables()["trials"] == 0
    g.close()


def test_edge_cases_and_errors():
    import paper_2106_05593_b200 as P
    with pytest.raises(P.MMCError):
        P.MMC(5, 4, 1, 5e-9, 5e-9, 5e-9, 0b001)                     # odd periodic length
    with pytest.raises(P.MMCError):
        P.MMC(0, 4, 1, 5e-9, 5e-9, 5e-9, 0)
    g = P.MMC(8, 8, 1, 5e-9, 5e-9, 5e-9, 0)
    with pytest.raises(P.MMCError):
        g.sweep(1)                                                  # nothing set
    g.set_material([P.Material(Ms0=8e5, A0=1.3e-11, Tc=870.0)]); g.set_temperature(300.0)
    with pytest.raises(P.MMCError) as e:
        g.set_m(np.zeros(64), np.zeros(64), np.zeros(64))           # zero-length non-empty cell (G13)
    assert e.value.code == -2
    with pytest.raises(P.MMCError):
        g.set_temperature(-1.0)
    g.close()
    # all cells empty: sweeps are no-ops, no trials
    g = P.MMC(8, 4, 2, 5e-9, 5e-9, 5e-9, 0)
    g.set_material([P.Material()]); g.set_temperature(300.0); g.set_m(np.zeros(64), np.zeros(64), np.zeros(64))
    g.sweep(3)
    ob = g.observables()
    assert ob["trials"] == 0 and ob["sweeps_done"] == 3
    g.close()
    # a 1x1x1 mesh: a single cell, no neighbours
    g = P.MMC(1, 1, 1, 5e-9, 5e-9, 5e-9, 0)
    g.set_material([P.Material(Ms0=8e5, A0=1.3e-11, Tc=870.0)]); g.set_temperature(300.0); g.set_move(20.0, -1.0, False)
    g.set_m([0.0], [0.0], [0.8675]); g.sweep(10)
    assert g.observables()["trials"] == 10
    g.close()
    # different A0 in two non-empty regions is outside the build
    g = P.MMC(8, 8, 1, 5e-9, 5e-9, 5e-9, 0)
    g.set_material([P.Material(Ms0=8e5, A0=1.3e-11, Tc=870.0), P.Material(Ms0=8e5, A0=1.0e-11, Tc=870.0)], np.arange(64) % 2)
    g.set_temperature(300.0)
    with pytest.raises(P.MMCError) as e:
        g.set_m(np.zeros(64), np.zeros(64), np.ones(64))
    assert e.value.code == -5
    g.close()


def test_state_check_and_buffer_growth_on_a_long_lived_context():
    """Host-side robustness of the boundary: (1) values in empty cells are ignored even when they are NaN markers (the library
    stores 0 there; 0-weights times NaN would otherwise poison every neighbour and the whole demag field); (2) |m| >= 2 is
    refused (m = M/Ms0; the pass's fixed-point sums are exact for |m| < 2); (3) a context whose class count shrinks and then
    grows with cubic anisotropy switched on in between re-allocates every table to its own size: the final state equals that
    of a fresh context configured directly."""
    import paper_2106_05593_b200 as P
    wl = W.cfg5(nx=160, ny=150)
    empty = wl.region_of_cell == 0
    m_nan = wl.m0.copy(); m_nan[:, empty] = np.nan
    a, b = _gpu(wl), _gpu(wl)
    a.set_m(*m_nan)
    a.sweep(3); b.sweep(3)
    ma, mb = a.get_m(), b.get_m()
    assert all(bool((ma[q] == mb[q]).all()) for q in range(3))
    assert all(bool((ma[q].cpu().numpy()[empty] == 0).all()) for q in range(3))
    oa, ob = a.observables(), b.observables()
    assert oa["accepted"] == ob["accepted"] and oa["E_demag"] == ob["E_demag"] and np.isfinite(oa["E_demag"])
    big = wl.m0.copy(); big[:, ~empty] *= 8.6e5
    with pytest.raises(P.MMCError) as e:
        a.set_m(*big)
    assert e.value.code == -1
    a.close(); b.close()
    # (3)
    nx, ny = 20, 16; N = nx * ny
    rng = np.random.default_rng(5)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (0.9 * v).astype(np.float32)
    plain = P.Material(Ms0=1.71e6, A0=2.1e-11, K1=4e4, Tc=1044.0)
    cubic = P.Material(Ms0=1.71e6, A0=2.1e-11, K1=4e4, Tc=1044.0, K1c=4.8e4, K2c=-1e4, K2=2e4, c1x=1.0, c1y=0.2, c1z=0.0, c2x=0.0, c2y=1.0, c2z=0.3)
    T100 = (300.0 + np.arange(N) % 100).astype(np.float32); T10 = (300.0 + np.arange(N) % 10).astype(np.float32)

    def ctx():
        g = P.MMC(nx, ny, 1, 2e-9, 2e-9, 2e-9, 0b011)
        g.set_move(25.0, -1.0, False); g.set_seed(11)
        return g
    g = ctx()
    g.set_material([plain]); g.set_temperature(300.0, T100); g.set_m(*m0); g.sweep(1)      # 100 classes, no cubic table
    g.set_material([cubic]); g.set_temperature(300.0, T10); g.set_m(*m0); g.sweep(1)       # 10 classes, cubic table of 10
    g.set_temperature(300.0, T100); g.set_m(*m0); g.set_sweep_counter(0); g.sweep(3)       # 100 classes WITH cubic
    h = ctx()
    h.set_material([cubic]); h.set_temperature(300.0, T100); h.set_m(*m0); h.sweep(3)
    mg, mh = g.get_m(), h.get_m()
    assert all(bool((mg[q] == mh[q]).all()) for q in range(3))
    assert g.observables()["E_an"] == h.observables()["E_an"]
    g.close(); h.close()


def test_adaptive_cone_tracks_oracle():
    """S11: same acceptance counts => same cone trajectory."""
    wl = W.cfg1(paper_regime=True); wl.adaptive_cone = True; wl.cone_deg = 30.0
    g, o = _gpu(wl), _orc(wl)
    g.sweep(300); o.run(300)
    og = g.observables()
    assert og["cone_deg"] == o.cone_deg and og["cone_deg"] < 30.0
    assert abs(og["accepted"] / og["trials"] - o.accepted / o.trials) < 5e-3
    g.close()


def test_relax_chunked_convergence():
    """mmc_relax against the oracle's driver of the same protocol on a small film:
    the same number of chunks, chunk averages within the trajectory noise of near-margin flips; and, exactly, against the
    library's own running averages of a second context driven by hand (integer fixed-point sums: bit-identical)."""
    wl = W.cfg2(nx=24, ny=20)
    wl.adaptive_cone = False
    g, o = _gpu(wl), _orc(wl)
    rg = g.relax((1.0, 0.0, 0.0), chunk_sweeps=20, min_chunks=2, max_chunks=5, threshold=5e-3)
    ro = o.relax((1.0, 0.0, 0.0), chunk_sweeps=20, min_chunks=2, max_chunks=5, threshold=5e-3)
    assert rg["chunks_done"] == ro["chunks_done"] and rg["converged"] == ro["converged"] and rg["sweeps"] == ro["sweeps"]
    assert abs(rg["mean_par_last"] - ro["mean_par_last"]) < 2e-4 and abs(rg["mean_len"] - ro["mean_len"]) < 2e-5
    h = _gpu(wl)
    for _ in range(rg["chunks_done"]):
        h.reset_averages(); h.sweep(20)
    ob = h.observables()
    assert np.array_equal(ob["run_mean_m"], rg["mean_m"]) and ob["run_mean_len"] == rg["mean_len"]
    # protocol edges: zero threshold never accepts; invalid arguments are refused
    r0 = g.relax((1.0, 0.0, 0.0), chunk_sweeps=3, min_chunks=2, max_chunks=3, threshold=0.0)
    assert (not r0["converged"]) and r0["chunks_done"] == 3 and r0["sweeps"] == 9
    import paper_2106_05593_b200 as P
    for bad in (dict(direction=(0, 0, 0)), dict(direction=(1, 0, 0), min_chunks=1), dict(direction=(1, 0, 0), chunk_sweeps=0)):
        with pytest.raises(P.MMCError):
            g.relax(**bad)
    g.close(); h.close()


@pytest.mark.parametrize("shape", [(256, 130, 1), (256, 66, 3), (1024, 65, 2), (140, 300, 4), (64, 48, 2)])
def test_demag_and_sweep_are_bitwise_reproducible(shape):
    """Race detector by determinism (compute-sanitizer is not available on the GPU pool): the hand-written transforms exchange
    data through shared memory between barriers, the pass reduces with integer atomics; any missing barrier or
    order-dependent sum would show up as run-to-run differences.  The same convolution 12 times, and two contexts running
    the same 30 iterations, must agree bit for bit."""
    import paper_2106_05593_b200 as P
    nx, ny, nz = shape; N = nx * ny * nz
    rng = np.random.default_rng(N + 1)
    v = rng.normal(size=(3, N)); v /= np.linalg.norm(v, axis=0)
    m0 = (0.8 * v).astype(np.float32)

    def make():
        g = P.MMC(nx, ny, nz, 3e-9, 3e-9, 3e-9, 0)
        g.set_material([P.Material(Ms0=8.6e5, A0=1.3e-11, K1=1e5, Tc=870.0)])
        g.set_temperature(500.0); g.set_move(20.0, -1.0, True); g.set_demag(True); g.set_seed(77); g.set_m(*m0)
        return g

    g = make()
    ref = [b.clone() for b in g.demag_field()]
    for _ in range(11):
        b = g.demag_field()
        assert all(bool((b[a] == ref[a]).all()) for a in range(3))
    h = make()
    g.sweep(30); h.sweep(30)
    mg, mh = g.get_m(), h.get_m()
    assert all(bool((mg[a] == mh[a]).all()) for a in range(3))
    og, oh = g.observables(), h.observables()
    for k in ("accepted", "trials", "run_mean_len", "E_ex", "E_demag", "cone_deg"):
        assert og[k] == oh[k], k
    assert np.array_equal(og["run_mean_m"], oh["run_mean_m"])
    g.close(); h.close()


@pytest.mark.parametrize("name", ["cfg2_64x48", "cfg4_30x21x3", "cfg1_32x32"])
def test_contexts_on_their_own_streams_agree_bitwise_with_the_default_stream(name):
    """Every call of the library is ordered on the stream given at mmc_create (graphs are captured on a private stream and
    launched into it): two contexts on two non-blocking streams, driven alternately without host synchronisation in between,
    end in the state of a context on the legacy default stream, bit for bit."""
    import paper_2106_05593_b200 as P
    wl = CASES[name]()
    ref = _gpu(wl); ref.sweep(40)
    mr = [t.clone() for t in ref.get_m()]; orf = ref.observables()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs = []
    for st in streams:
        with torch.cuda.stream(st):
            c = P.MMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, stream=st)
            W.configure(c, wl, P.Material)
            ctxs.append(c)
    for chunk in (1, 17, 3, 19):                     # plain launches, graphs of 16 and of 1 iteration; alternating contexts
        for c, st in zip(ctxs, streams):
            with torch.cuda.stream(st):
                c.sweep(chunk)
    for c, st in zip(ctxs, streams):
        with torch.cuda.stream(st):
            m = c.get_m(); ob = c.observables()      # synchronises the context's stream
            assert all(torch.equal(m[q], mr[q]) for q in range(3))
            for k in ("accepted", "trials", "sweeps_done", "cone_deg", "run_mean_len", "E_ex", "E_demag", "E_long"):
                assert ob[k] == orf[k], k
        c.close()
    ref.close()


@pytest.mark.parametrize("name", ["cfg2_64x48", "cfg3_64x64_200K", "cfg4_30x21x3", "cfg5_160x150"])
def test_launch_paths_agree_bitwise(name):
    """mmc_sweep(n) replays whole iterations from CUDA graphs (16 at a time, then one at a time), and on small meshes the last
    CTA of the black pass closes the iteration.  Plain stream launches (MMC_NO_GRAPH), kernels chained by programmatic
    dependent launch (MMC_PDL=1: an option, measured slower) and the event-bracketed launches of
    mmc_sweep_timed must give the same bits: states, counters, cone, running sums after 137 iterations with the adaptive cone
    (one controller window and a partial one; 8 x 16 + 9 iterations; a second call re-uses the cached graphs)."""
    ref = None
    for knob in (None, "MMC_NO_GRAPH", "MMC_PDL", "timed"):
        wl = CASES[name](); wl.adaptive_cone = True
        import contextlib
        with (_env(knob, "1") if knob and knob != "timed" else contextlib.nullcontext()):
            g = _gpu(wl)
            if knob == "timed":
                g.sweep_timed(100); g.sweep_timed(37)
            else:
                g.sweep(100); g.sweep(37)
            m = [x.clone() for x in g.get_m()]; ob = g.observables()
            g.close()
        if ref is None:
            ref = (m, ob)
            continue
        assert all(bool((m[q] == ref[0][q]).all()) for q in range(3)), knob
        for k in ("accepted", "trials", "sweeps_done", "cone_deg", "run_sweeps", "run_mean_len", "E_ex", "E_demag"):
            assert ob[k] == ref[1][k], (knob, k)
        assert np.array_equal(ob["run_mean_m"], ref[1]["run_mean_m"]), knob
    assert ref[1]["sweeps_done"] == 137


@pytest.mark.parametrize("name", ["cfg3_64x64_200K", "cfg4_30x21x3", "cfg5_160x150"])
def test_histograms_parity(name):
    """mmc_histogram against the oracle's histograms of the same seeded state: integer
    counts, both sides deciding the bin in fp64 from the fp32 state.  Bit-exact for the length histogram; the angle histogram
    goes through acos and a mean direction summed in a different order (1e-16 relative), so a count may move between
    NEIGHBOURING bins for a value within ~1e-15 of an edge: none is expected and none is tolerated beyond that."""
    wl = CASES[name]()
    g, o = _gpu(wl), _orc(wl)
    rng = np.random.default_rng(11)
    v = rng.normal(size=(3, wl.N)); v /= np.linalg.norm(v, axis=0)
    v[0] = np.abs(v[0]) + 0.2
    m0 = (rng.uniform(0.05, 1.1, wl.N) * v).astype(np.float32)
    g.set_m(*m0); o.set_m(*m0)
    for nb, lo, hi in ((100, 0.0, 1.2), (37, 0.3, 0.9), (1, 0.0, 2.0), (4096, 0.05, 1.1)):
        cg, ug, og_ = g.histogram("length", nb, lo, hi)
        co, uo, oo = o.histogram("length", nb, lo, hi)
        assert np.array_equal(cg, co) and ug == uo and og_ == oo
        assert int(cg.sum()) + ug + og_ == wl.n_active
    for nb, lo, hi in ((100, 0.0, np.pi), (100, 0.2, 2.0)):
        cg, ug, og_ = g.histogram("angle", nb, lo, hi)
        co, uo, oo = o.histogram("angle", nb, lo, hi)
        assert int(cg.sum()) + ug + og_ == wl.n_active
        diff = cg.astype(np.int64) - co.astype(np.int64)
        assert np.abs(diff).sum() <= 2 and diff.sum() == (uo + oo) - (ug + og_)
    import paper_2106_05593_b200 as P
    with pytest.raises(P.MMCError):
        g.histogram("length", 0, 0.0, 1.0)
    with pytest.raises(P.MMCError):
        g.histogram("length", 10, 1.0, 1.0)
    g.close()


@pytest.mark.parametrize("name", ["cfg1_32x32", "cfg1_paper_regime", "cfg1_ragged_40x24", "cfg1_ragged_periodic_12x6", "cfg1_k2_32x32",
                                  "cfg1_64x48_loop_kernel", "cfg1_periodic_2x6", "cfg4_nodemag_periodic_16x12x4", "cfg4_nodemag_24x20x4",
                                  "cfg4_nodemag_periodic_z_15x9x2", "cfg5_nodemag_90x80"])
def test_single_launch_small_mesh_path_is_bitwise_the_launch_per_pass_path(name):
    """Small meshes without demag run all iterations of mmc_sweep in ONE launch (one CTA, SURVEY 8(d) "Config 1"); mmc_sweep_timed
    keeps the launch-per-pass kernels.  Same cell arithmetic, integer reductions: states, counters, energies and the
    adaptive cone must agree bit for bit after 230 iterations (two cone-controller windows and a partial one)."""
    # <= 512 cells per colour: the pipelined kernel (one thread per cell, the two colours' half updates overlap); more: the loop kernel
    extra = {"cfg1_64x48_loop_kernel": lambda: W.cfg1(nx=64, ny=48, paper_regime=True),
             # several layers, per-cell classes, empty cells: the recipes of configs 4 and 5 with the demag term switched off
             "cfg4_nodemag_periodic_16x12x4": lambda: _with_pbc(W.cfg4(nx=16, ny=12, nz=4), 0b111),
             "cfg4_nodemag_24x20x4": lambda: W.cfg4(nx=24, ny=20, nz=4),
             "cfg4_nodemag_periodic_z_15x9x2": lambda: _with_pbc(W.cfg4(nx=15, ny=9, nz=2), 0b100),
             "cfg5_nodemag_90x80": lambda: W.cfg5(nx=90, ny=80)}
    wl = extra[name]() if name in extra else CASES[name]()
    wl.demag = False
    wl.adaptive_cone = True
    a, b = _gpu(wl), _gpu(wl)
    a.sweep(230)
    b.sweep_timed(230)
    ma, mb = a.get_m(), b.get_m()
    assert all(bool((ma[q] == mb[q]).all()) for q in range(3))
    oa, ob = a.observables(), b.observables()
    for k in ("accepted", "trials", "sweeps_done", "cone_deg", "run_sweeps", "E_ex", "E_an", "E_long"):
        assert oa[k] == ob[k], k
    # running means: both paths add 2^-22 fixed-point values; the launch-per-pass kernel rounds the sum of a thread's two
    # cells, this one every cell: they agree to that quantum
    assert abs(oa["run_mean_len"] - ob["run_mean_len"]) < 2.0 ** -22 and np.abs(oa["run_mean_m"] - ob["run_mean_m"]).max() < 2.0 ** -22
    assert oa["sweeps_done"] == 230
    a.close(); b.close()
