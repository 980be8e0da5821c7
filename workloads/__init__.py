"""Seeded synthetic workloads shaped like BASELINE.json's five configs ("input recipe").

This module serves BOTH the oracle and the CUDA path and therefore holds none of the method's
arithmetic: no thermal functions, no energies, no RNG of the method, no demag.  It only draws
geometry / material tables / initial vectors with numpy's PCG64 and hands them to any simulator
object exposing the setter names of include/mmc.h (``configure``).  Initial lengths |m0| are plain
recipe numbers (quoted in DESIGN.md), not computed from Eq. (9).

The paper measures on no public dataset; its workloads are synthetic geometries (ellipse
PAPER.md:133, Voronoi film PAPER.md:145, Co/Pt film PAPER.md:158, ASI PAPER.md:184) and these
stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

MUB = 9.2740100783e-24
BASE_SEED = 20210605 * 100


@dataclass
class Workload:
    name: str
    nx: int; ny: int; nz: int
    dx: float; dy: float; dz: float
    pbc_mask: int
    regions: list                      # list of dict(Ms0,A0,K1,ax,ay,az,D0,Tc,mu_atom)
    region_of_cell: np.ndarray | None  # int32[N] or None (all region 0)
    inter_region_exchange: int
    T_uniform: float
    T_per_cell: np.ndarray | None      # float32[N] or None
    B_ext: tuple
    cone_deg: float
    sigma: float                       # < 0 => Eq. (13) with the 0.03 cap
    adaptive_cone: bool
    demag: bool
    seed: int
    m0: np.ndarray                     # float32[3, N]
    schedule: list = field(default_factory=list)   # [(kind, value, n_sweeps)], kind in {"B","T"}
    demag_updates: int = 1

    @property
    def N(self):
        return self.nx * self.ny * self.nz

    @property
    def n_active(self):
        if self.region_of_cell is None:
            return self.N if self.regions[0]["Ms0"] > 0 else 0
        ms = np.array([r["Ms0"] for r in self.regions])
        return int((ms[self.region_of_cell] > 0).sum())


def _mat(Ms0=0.0, A0=0.0, K1=0.0, axis=(0.0, 0.0, 1.0), D0=0.0, Tc=1.0, mu_atom=MUB, K1c=0.0, K2c=0.0,
         c1=(1.0, 0.0, 0.0), c2=(0.0, 1.0, 0.0)):
    d = dict(Ms0=Ms0, A0=A0, K1=K1, ax=axis[0], ay=axis[1], az=axis[2], D0=D0, Tc=Tc, mu_atom=mu_atom)
    if K1c != 0.0 or K2c != 0.0:                     # cubic anisotropy, Eq. (12): two of the cubic axes
        d.update(K1c=K1c, K2c=K2c, c1x=c1[0], c1y=c1[1], c1z=c1[2], c2x=c2[0], c2y=c2[1], c2z=c2[2])
    return d


def _random_unit(rng, n):
    z = rng.uniform(-1.0, 1.0, n); ph = rng.uniform(0.0, 2 * np.pi, n)
    s = np.sqrt(1.0 - z * z)
    return np.stack([s * np.cos(ph), s * np.sin(ph), z])


def configure(sim, wl: Workload, material_cls=None):
    """Push a workload through the setter names shared by include/mmc.h's binding and the oracle.
    ``material_cls`` builds one region record from keyword arguments (each side has its own)."""
    regs = [material_cls(**r) for r in wl.regions] if material_cls else wl.regions
    sim.set_material(regs, wl.region_of_cell)
    sim.set_exchange_coupling(wl.inter_region_exchange)
    sim.set_temperature(wl.T_uniform, wl.T_per_cell)
    sim.set_field(*wl.B_ext)
    sim.set_move(wl.cone_deg, wl.sigma, wl.adaptive_cone)
    sim.set_demag(wl.demag, wl.demag_updates)
    sim.set_seed(wl.seed)
    sim.set_sweep_counter(0)
    sim.set_m(wl.m0[0], wl.m0[1], wl.m0[2])
    return sim


# ------------------------------------------------------------------------------------------------
def cfg1(nx=32, ny=32, paper_regime=False):
    """Tiny film, no demag: 32x32x1, 5 nm, PBC x/y, Ms0 8e5, A 1.3e-11, K1 5e5 || z, Tc 870, 300 K,
    cone 30 deg fixed, length factor 1 + U[-0.05, 0.05], random unit vectors x 0.8675 (~me(300 K))."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 1))
    m0 = (0.86750232 * _random_unit(rng, nx * ny)).astype(np.float32)
    cone, sig = (8.0, -1.0) if paper_regime else (30.0, 0.05)
    return Workload("cfg1_tiny_film" + ("_paper_regime" if paper_regime else ""), nx, ny, 1, 5e-9, 5e-9, 5e-9, 0b011,
                    [_mat(8e5, 1.3e-11, 5e5, (0, 0, 1), 0.0, 870.0)], None, 1, 300.0, None, (0.0, 0.0, 0.0),
                    cone, sig, False, False, BASE_SEED + 1, m0, [("B", (0.0, 0.0, 0.0), 1000)])


def cfg2(nx=256, ny=256):
    """Demag film with field sweep: 256x256x1, 5 nm, open, permalloy-like, 300 K, start saturated +x,
    B_x from +100 mT to -100 mT in 2 mT steps, 200 sweeps/step, adaptive cone from 30 deg, Eq. (13) sigma."""
    N = nx * ny
    m0 = np.zeros((3, N), dtype=np.float32); m0[0] = 0.8675
    sched = [("B", (1e-3 * b, 0.0, 0.0), 200) for b in range(100, -101, -2)]
    return Workload("cfg2_demag_film", nx, ny, 1, 5e-9, 5e-9, 5e-9, 0,
                    [_mat(8.6e5, 1.3e-11, 0.0, (0, 0, 1), 0.0, 870.0)], None, 1, 300.0, None, (0.1, 0.0, 0.0),
                    30.0, -1.0, True, True, BASE_SEED + 2, m0, sched)


def cfg3(nx=512, ny=512, T=200.0):
    """Chiral film: 512x512x1, 2 nm, PBC x/y for exchange+DMI, Ms0 6e5, A 1e-11, K1 8e5 || z,
    D 2.5e-3, Tc 700, open-boundary Newell demag, B_z 100 mT, T from 200 K to 800 K in 50 K steps,
    5000 sweeps per T, random start at |m| = 0.8934 (~me(200 K))."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 3))
    m0 = (0.89339791 * _random_unit(rng, nx * ny)).astype(np.float32)
    sched = [("T", float(t), 5000) for t in range(200, 801, 50)]
    return Workload("cfg3_chiral_film", nx, ny, 1, 2e-9, 2e-9, 2e-9, 0b011,
                    [_mat(6e5, 1e-11, 8e5, (0, 0, 1), 2.5e-3, 700.0)], None, 1, T, None, (0.0, 0.0, 0.1),
                    30.0, -1.0, True, True, BASE_SEED + 3, m0, sched)


def cfg4(nx=1024, ny=1024, nz=4):
    """Granular medium: 3 nm cells, 3-D Poisson-Voronoi grains of mean diameter 8 nm (one region per
    grain, no exchange between grains), per-grain axis uniform on a 5 deg cap about z, K1 3e6,
    per-grain Tc ~ N(700 K, 21 K), Gaussian hot spot FWHM 20 nm (750 K peak on 300 K), demag,
    Ms0 1.1e6 and A0 1e-11 (FePt-like fillers; BASELINE.json gives none), open boundaries, B = 0,
    start along +axis at |m0| = max(0.02, sqrt(max(0, 1 - T/Tc)))."""
    from scipy.spatial import cKDTree
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 4))
    h = 3.0  # nm
    vol = nx * ny * nz * h ** 3
    n_seeds = max(2, int(round(vol / (np.pi * 8.0 ** 3 / 6.0))))
    seeds = rng.uniform(0.0, 1.0, (n_seeds, 3)) * np.array([nx * h, ny * h, nz * h])
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    pts = np.stack([(i.ravel() + 0.5) * h, (j.ravel() + 0.5) * h, (k.ravel() + 0.5) * h], axis=1)
    _, grain = cKDTree(seeds).query(pts, workers=-1)
    grain = grain.astype(np.int32)
    cosmin = np.cos(np.deg2rad(5.0))
    cz = rng.uniform(cosmin, 1.0, n_seeds); ph = rng.uniform(0, 2 * np.pi, n_seeds); s = np.sqrt(1 - cz * cz)
    axes = np.stack([s * np.cos(ph), s * np.sin(ph), cz], axis=1)
    Tc = rng.normal(700.0, 21.0, n_seeds)
    regions = [_mat(1.1e6, 1e-11, 3e6, tuple(axes[g]), 0.0, float(Tc[g])) for g in range(n_seeds)]
    x = (i.ravel() + 0.5) * h - 0.5 * nx * h; y = (j.ravel() + 0.5) * h - 0.5 * ny * h
    T = (300.0 + 450.0 * np.exp(-4.0 * np.log(2.0) * (x * x + y * y) / 20.0 ** 2)).astype(np.float32)
    L = np.maximum(0.02, np.sqrt(np.maximum(0.0, 1.0 - T.astype(np.float64) / Tc[grain])))
    m0 = (axes[grain].T * L).astype(np.float32)
    return Workload("cfg4_granular", nx, ny, nz, 3e-9, 3e-9, 3e-9, 0, regions, grain, 0, 300.0, T,
                    (0.0, 0.0, 0.0), 30.0, -1.0, True, True, BASE_SEED + 4, m0, [("B", (0.0, 0.0, 0.0), 2000)])


def cfg5(nx=2048, ny=2048):
    """Artificial spin ice: 5x5x10 nm cells, stadium islands 50x16 cells on a 70-cell square lattice
    (horizontal islands centred at ((p+1/2)a, qa), vertical at (pa, (q+1/2)a)), only islands wholly
    inside the mesh, empty elsewhere; Ms0 8.6e5, A 1.3e-11, K1 0, Tc 870, 500 K, demag, field along
    [11] from 0 to 50 mT in 2 mT steps, 500 sweeps/step, start along the long axis at |m| = 0.743."""
    a, Lh, Wh = 70, 25.0, 8.0
    j, i = np.meshgrid(np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    mask = np.zeros((ny, nx), dtype=np.int32)
    m0 = np.zeros((3, ny, nx), dtype=np.float32)

    def stadium(cx, cy, horizontal):
        u, v = (i - cx, j - cy) if horizontal else (j - cy, i - cx)
        du = np.maximum(np.abs(u) - (Lh - Wh), 0.0)
        return du * du + v * v <= Wh * Wh

    for q in range(0, ny // a + 2):
        for p in range(0, nx // a + 2):
            cx, cy = (p + 0.5) * a, q * a            # horizontal island
            if cx - Lh >= 0 and cx + Lh <= nx and cy - Wh >= 0 and cy + Wh <= ny:
                sel = stadium(cx, cy, True); mask[sel] = 1; m0[0][sel] = 0.74303265
            cx, cy = p * a, (q + 0.5) * a            # vertical island
            if cx - Wh >= 0 and cx + Wh <= nx and cy - Lh >= 0 and cy + Lh <= ny:
                sel = stadium(cx, cy, False); mask[sel] = 1; m0[1][sel] = 0.74303265
    s = 1.0 / np.sqrt(2.0)
    sched = [("B", (1e-3 * b * s, 1e-3 * b * s, 0.0), 500) for b in range(0, 51, 2)]
    return Workload("cfg5_spin_ice", nx, ny, 1, 5e-9, 5e-9, 10e-9, 0,
                    [_mat(), _mat(8.6e5, 1.3e-11, 0.0, (0, 0, 1), 0.0, 870.0)], mask.ravel(), 1, 500.0, None,
                    (0.0, 0.0, 0.0), 30.0, -1.0, True, True, BASE_SEED + 5, m0.reshape(3, -1), sched)


CONFIGS = {1: cfg1, 2: cfg2, 3: cfg3, 4: cfg4, 5: cfg5}


def fe_film(nx=400, ny=400, nz=10):
    """The paper's granular Fe film with cubic anisotropy (Fig. 5; SURVEY 8(f) row 3's workload): 2 nm cubic
    cells, periodic in the plane (exchange; the demag convolution is open-boundary as everywhere), Ms0 1.71e6, A0 2.1e-11,
    K1c 4.8e4, K2c -1e4 (4th / 6th order), Tc 1044, T 300 K; 3-D Voronoi grains with 10 nm mean seed spacing and phase
    separation (no exchange between grains); field along +x.  Filler the paper leaves open: each grain's cubic axes are a
    random rotation (seeded); start saturated along +x at |m0| = 0.97 (~me(300 K))."""
    from scipy.spatial import cKDTree
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 6))
    h = 2.0
    n_seeds = max(2, int(round(nx * ny * nz * h ** 3 / 10.0 ** 3)))
    seeds = rng.uniform(0.0, 1.0, (n_seeds, 3)) * np.array([nx * h, ny * h, nz * h])
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    pts = np.stack([(i.ravel() + 0.5) * h, (j.ravel() + 0.5) * h, (k.ravel() + 0.5) * h], axis=1)
    _, grain = cKDTree(seeds).query(pts, workers=-1)
    grain = grain.astype(np.int32)
    regions = []
    for g in range(n_seeds):
        q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
        regions.append(_mat(1.71e6, 2.1e-11, 0.0, (0.0, 0.0, 1.0), 0.0, 1044.0, K1c=4.8e4, K2c=-1.0e4,
                            c1=tuple(q[:, 0]), c2=tuple(q[:, 1])))
    N = nx * ny * nz
    m0 = np.zeros((3, N), dtype=np.float32); m0[0] = 0.97
    sched = [("B", (1e-3 * b, 0.0, 0.0), 2000) for b in range(-200, 201, 10)]
    return Workload("fe_film_cubic", nx, ny, nz, 2e-9, 2e-9, 2e-9, 0b011, regions, grain, 0, 300.0, None,
                    (0.05, 0.0, 0.0), 30.0, -1.0, True, True, BASE_SEED + 6, m0, sched)


CONFIGS[6] = fe_film


def make(cfg: int, **kw) -> Workload:
    return CONFIGS[cfg](**kw)
