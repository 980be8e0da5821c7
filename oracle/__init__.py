"""fp64 CPU oracle for the MMC hot path of arXiv:2106.05593 -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_2106_05593_b200`` (the CUDA path)
and neither imports the other.  The arithmetic lives in ``mmc_oracle.c`` (plain C, fp64, one cell
at a time, the paper's order); this module only builds it with gcc, marshals numpy arrays, does the
per-class thermal set-up bookkeeping, and provides the zero-padded FFT convolution of Eq. (14) with
``numpy.fft`` as the library step.

Parity pins (tests/test_oracle_*.py, ``-m "not gpu"``): Philox known answers; thermal functions vs
series / Curie-Weiss / SURVEY probe values; trial-move geometry; single-cell Langevin <cos> and
length-distribution quadrature; local dF == global dE by brute force; detailed-balance ratio;
colour-order independence; Newell invariants + independent 6-D quadrature; FFT == direct sum.
Unpinned (stated in DESIGN.md): equilibrium of coupled meshes with exchange+DMI+demag against any
external value -- "parity unpinned" for that item only.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mmc_oracle.c")
_LIB = os.path.join(_HERE, "libmmc_oracle.so")

KB = 1.380649e-23
MU0 = 4e-7 * np.pi
MUB = 9.2740100783e-24


def build(force: bool = False) -> str:
    """Compile mmc_oracle.c with gcc (-O2, OpenMP, libquadmath).  Building is not using."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               _SRC, "-o", _LIB, "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("pbc", C.c_uint32),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("active", C.c_void_p), ("region", C.c_void_p), ("inter_region_exchange", C.c_int32),
        ("Ms0", C.c_void_p), ("beta", C.c_void_p),
        ("c2", C.c_void_p), ("c4", C.c_void_p), ("c0", C.c_void_p),
        ("Kq", C.c_void_p), ("K1T", C.c_void_p),
        ("ax", C.c_void_p), ("ay", C.c_void_p), ("az", C.c_void_p),
        ("sigma", C.c_void_p),
        ("A0", C.c_double), ("D0", C.c_double), ("Bext", C.c_double * 3),
        ("bdx", C.c_void_p), ("bdy", C.c_void_p), ("bdz", C.c_void_p),
        ("one_minus_cos_cone", C.c_double), ("seed", C.c_uint64),
        ("K1cT", C.c_void_p), ("K2cT", C.c_void_p), ("cub", C.c_void_p),
        ("K2T", C.c_void_p), ("me2", C.c_void_p),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_u01.restype = C.c_double; L.orc_u01.argtypes = [C.c_uint32]
        L.orc_cell_uniforms.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, dp]
        for name in ("orc_langevin", "orc_langevin_prime"):
            getattr(L, name).restype = C.c_double; getattr(L, name).argtypes = [C.c_double]
        L.orc_me.restype = C.c_double; L.orc_me.argtypes = [C.c_double, C.c_double]
        L.orc_chi_par.restype = C.c_double; L.orc_chi_par.argtypes = [C.c_double] * 4
        L.orc_thermal.restype = C.c_int; L.orc_thermal.argtypes = [C.c_double] * 5 + [dp]
        L.orc_trial.argtypes = [dp, dp, C.c_double, C.c_double, dp, dp]
        L.orc_cell_dF.argtypes = [C.POINTER(_Problem), dp, dp, dp, C.c_int, C.c_int, C.c_int, dp, dp]
        L.orc_colour_pass.restype = C.c_int64
        L.orc_colour_pass.argtypes = [C.POINTER(_Problem), dp, dp, dp, C.c_int, C.c_uint64,
                                      C.c_void_p, C.c_int64, C.c_int,
                                      C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
        L.orc_colour_terms_given_dm.argtypes = [C.POINTER(_Problem), dp, dp, dp, C.c_int, dp, dp]
        L.orc_observables.argtypes = [C.POINTER(_Problem), dp, dp, dp, dp, dp, C.POINTER(C.c_int64)]
        L.orc_newell.argtypes = [C.c_double] * 6 + [dp]
        L.orc_demag_tensor.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [C.c_int, dp]
        L.orc_demag_direct.argtypes = [C.c_int] * 3 + [dp] * 7
        L.orc_exact_demag_dF.restype = C.c_double
        L.orc_exact_demag_dF.argtypes = [C.POINTER(_Problem)] + [dp] * 4 + [C.c_int64, dp]
        L.orc_serial_exact_sweep.restype = C.c_int64
        L.orc_serial_exact_sweep.argtypes = [C.POINTER(_Problem)] + [dp] * 7 + [C.c_uint64, C.c_int, C.POINTER(C.c_int64)]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


# ----------------------------------------------------------------------------- scalar helpers
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def u01(x: int) -> float:
    return lib().orc_u01(x)


def cell_uniforms(seed: int, sweep: int, cell: int):
    u = np.zeros(4)
    lib().orc_cell_uniforms(seed, sweep, cell, _dp(u))
    return u


def langevin(x): return lib().orc_langevin(float(x))
def langevin_prime(x): return lib().orc_langevin_prime(float(x))
def me_of_T(T, Tc): return lib().orc_me(float(T), float(Tc))
def chi_par(T, Tc, mu, me): return lib().orc_chi_par(float(T), float(Tc), float(mu), float(me))


def thermal(T, Tc, mu, V, Ms0):
    """-> dict(me, chi, c2, c4, c0, sigma13); Eq. (7),(8),(9),(13)."""
    o = np.zeros(6)
    if lib().orc_thermal(float(T), float(Tc), float(mu), float(V), float(Ms0), _dp(o)) != 0:
        raise ValueError("T must be > 0")
    return dict(me=o[0], chi=o[1], c2=o[2], c4=o[3], c0=o[4], sigma13=o[5])


def trial(m, u3, one_minus_cos_cone, sigma):
    m = np.ascontiguousarray(m, dtype=np.float64); u3 = np.ascontiguousarray(u3, dtype=np.float64)
    dm = np.zeros(3); f = C.c_double()
    lib().orc_trial(_dp(m), _dp(u3), float(one_minus_cos_cone), float(sigma), _dp(dm), C.byref(f))
    return dm, f.value


def newell(X, Y, Z, dx, dy, dz):
    o = np.zeros(6)
    lib().orc_newell(float(X), float(Y), float(Z), float(dx), float(dy), float(dz), _dp(o))
    return o


def demag_tensor(nx, ny, nz, dx, dy, dz, r_near=32):
    """Octant table [6, nz, ny, nx] (xx,yy,zz,xy,xz,yz) for offsets >= 0."""
    out = np.zeros((6, nz, ny, nx))
    lib().orc_demag_tensor(nx, ny, nz, float(dx), float(dy), float(dz), int(r_near), _dp(out))
    return out


def demag_direct(tab, Mx, My, Mz):
    """B_d = -mu0 sum_j N(r_i-r_j) M_j by the O(N^2) sum (Eq. (14)); arrays shaped [nz, ny, nx]."""
    _, nz, ny, nx = tab.shape
    Mx, My, Mz = (np.ascontiguousarray(a, dtype=np.float64) for a in (Mx, My, Mz))
    b = [np.zeros((nz, ny, nx)) for _ in range(3)]
    lib().orc_demag_direct(nx, ny, nz, _dp(tab), _dp(Mx), _dp(My), _dp(Mz), _dp(b[0]), _dp(b[1]), _dp(b[2]))
    return b


def _full_kernel(tab):
    """Place the octant table on the zero-padded periodic grid: offset o_d, |o_d|<N_d,
    stored at index o_d mod P_d, P_d = 2 N_d (P_d = 1 when N_d = 1); index N_d left zero.  Diagonal
    components are even in every coordinate, N_ab (a != b) is odd in coordinates a and b."""
    _, nz, ny, nx = tab.shape
    P = [1 if n == 1 else 2 * n for n in (nz, ny, nx)]
    full = np.zeros((6, P[0], P[1], P[2]))
    par = {0: (1, 1, 1), 1: (1, 1, 1), 2: (1, 1, 1), 3: (1, -1, -1), 4: (-1, 1, -1), 5: (-1, -1, 1)}  # (z,y,x) signs
    for sz_ in ((1, -1) if nz > 1 else (1,)):
        for sy_ in ((1, -1) if ny > 1 else (1,)):
            for sx_ in ((1, -1) if nx > 1 else (1,)):
                oz = np.arange(nz) if sz_ > 0 else np.arange(1, nz)
                oy = np.arange(ny) if sy_ > 0 else np.arange(1, ny)
                ox = np.arange(nx) if sx_ > 0 else np.arange(1, nx)
                if oz.size == 0 or oy.size == 0 or ox.size == 0:
                    continue
                for q in range(6):
                    pz, py, px = par[q]
                    sgn = (pz if sz_ < 0 else 1) * (py if sy_ < 0 else 1) * (px if sx_ < 0 else 1)
                    full[q][np.ix_((sz_ * oz) % P[0], (sy_ * oy) % P[1], (sx_ * ox) % P[2])] = sgn * tab[q][np.ix_(oz, oy, ox)]
    return full


class DemagFFT:
    """Zero-padded FFT convolution of Eq. (14) in fp64 with numpy.fft."""

    def __init__(self, nx, ny, nz, dx, dy, dz, r_near=32):
        self.shape = (nz, ny, nx)
        self.tab = demag_tensor(nx, ny, nz, dx, dy, dz, r_near)
        full = _full_kernel(self.tab)
        self.P = full.shape[1:]
        self.Khat = np.fft.rfftn(full, axes=(1, 2, 3))

    def field(self, Mx, My, Mz):
        """B_d (tesla), arrays [nz, ny, nx]; M = Ms0 m in A/m, zero in empty cells."""
        nz, ny, nx = self.shape
        Mh = []
        for a in (Mx, My, Mz):
            pad = np.zeros(self.P); pad[:nz, :ny, :nx] = a
            Mh.append(np.fft.rfftn(pad))
        K = self.Khat
        Hx = -(K[0] * Mh[0] + K[3] * Mh[1] + K[4] * Mh[2])
        Hy = -(K[3] * Mh[0] + K[1] * Mh[1] + K[5] * Mh[2])
        Hz = -(K[4] * Mh[0] + K[5] * Mh[1] + K[2] * Mh[2])
        return [MU0 * np.fft.irfftn(H, s=self.P, axes=(0, 1, 2))[:nz, :ny, :nx] for H in (Hx, Hy, Hz)]


# ----------------------------------------------------------------------------- the MMC oracle
@dataclass
class Material:
    Ms0: float = 0.0; A0: float = 0.0; K1: float = 0.0
    ax: float = 0.0; ay: float = 0.0; az: float = 1.0
    D0: float = 0.0; Tc: float = 1.0; mu_atom: float = MUB
    # cubic anisotropy, Eq. (12): 4th and 6th order constants (J/m^3) and two of the cubic axes (the third is their cross
    # product; orthonormalised by Gram-Schmidt)
    K1c: float = 0.0; K2c: float = 0.0
    c1x: float = 1.0; c1y: float = 0.0; c1z: float = 0.0
    c2x: float = 0.0; c2y: float = 1.0; c2z: float = 0.0
    K2: float = 0.0          # 4th-order uniaxial constant of Eq. (11), J/m^3, same axis as K1


def cubic_axes(r):
    """The three orthonormal cubic axes of a region record as 9 numbers: e1 = c1/|c1|, e2 = the part of c2 orthogonal
    to e1, normalised, e3 = e1 x e2."""
    e1 = np.array([r.c1x, r.c1y, r.c1z], dtype=np.float64); e1 /= np.linalg.norm(e1)
    e2 = np.array([r.c2x, r.c2y, r.c2z], dtype=np.float64); e2 -= (e2 @ e1) * e1; e2 /= np.linalg.norm(e2)
    return np.concatenate([e1, e2, np.cross(e1, e2)])


class OracleMMC:
    """Step-by-step fp64 MMC.  State m is kept in float64; with
    ``store_fp32=True`` accepted vectors are rounded to fp32, the GPU's storage format."""

    def __init__(self, nx, ny, nz, dx, dy, dz, pbc_mask=0, store_fp32=True):
        self.nx, self.ny, self.nz = nx, ny, nz
        self.dx, self.dy, self.dz = dx, dy, dz
        self.pbc = pbc_mask
        for a, n in enumerate((nx, ny, nz)):
            if (pbc_mask >> a) & 1 and n % 2:
                raise ValueError("periodic dimension must have even length (O6)")
        self.N = nx * ny * nz
        self.V = dx * dy * dz
        self.store_fp32 = store_fp32
        self.regions = [Material()]
        self.region_of_cell = np.zeros(self.N, dtype=np.int32)
        self.inter_region_exchange = 1
        self.T_cell = np.full(self.N, 300.0)
        self.Bext = np.zeros(3)
        self.cone_deg = 30.0
        self.sigma_user = -1.0
        self.adaptive = False
        self.demag_enabled = False
        self.demag_updates = 1
        self.demag_r_near = 32
        self._demag = None
        self.has_cubic = False
        self.has_k2 = False
        self.seed = 0
        self.sweep = 0
        self.accepted = 0; self.trials = 0
        self._win_acc = 0; self._win_tri = 0; self._win_sweeps = 0
        self.m = [np.zeros(self.N) for _ in range(3)]
        self.bd = None
        self._dirty = True

    # -- set-up ---------------------------------------------------------------------------
    def set_material(self, regions, region_of_cell=None):
        self.regions = list(regions)
        self.region_of_cell = (np.zeros(self.N, dtype=np.int32) if region_of_cell is None
                               else np.ascontiguousarray(region_of_cell, dtype=np.int32).ravel())
        self._dirty = True

    def set_exchange_coupling(self, inter_region_exchange):
        self.inter_region_exchange = int(inter_region_exchange); self._dirty = True

    def set_temperature(self, T_uniform, T_per_cell=None):
        self.T_cell = (np.full(self.N, float(T_uniform)) if T_per_cell is None
                       else np.ascontiguousarray(T_per_cell, dtype=np.float32).astype(np.float64).ravel())
        self._dirty = True

    def set_field(self, Bx, By, Bz):
        self.Bext = np.array([Bx, By, Bz], dtype=np.float64)

    def set_move(self, cone_deg, sigma=-1.0, adaptive_cone=False):
        self.cone_deg = float(cone_deg); self.sigma_user = float(sigma); self.adaptive = bool(adaptive_cone)
        self._dirty = True

    def set_demag(self, enabled, updates_per_sweep=1, r_near=32):
        self.demag_enabled = bool(enabled); self.demag_updates = int(updates_per_sweep)
        self.demag_r_near = r_near

    def set_seed(self, seed): self.seed = int(seed)
    def set_sweep_counter(self, s): self.sweep = int(s)

    def set_m(self, mx, my, mz):
        self.m = [np.ascontiguousarray(np.asarray(a, dtype=np.float32).astype(np.float64).ravel()) for a in (mx, my, mz)]

    def get_m(self):
        return [a.copy() for a in self.m]

    def _setup(self):
        """O1: per-cell coefficients; one thermal solve per distinct (region, T) class."""
        if not self._dirty:
            return
        N = self.N
        reg = self.region_of_cell
        Ms0r = np.array([r.Ms0 for r in self.regions])
        self.active = np.ascontiguousarray((Ms0r[reg] > 0).astype(np.uint8))
        act_regs = [r for r in self.regions if r.Ms0 > 0]
        A0s = {r.A0 for r in act_regs}; D0s = {r.D0 for r in act_regs}
        if len(A0s) > 1 or len(D0s) > 1:
            raise ValueError("A0 and D0 must be uniform over non-empty regions")
        self.A0 = A0s.pop() if A0s else 0.0
        self.D0 = D0s.pop() if D0s else 0.0
        names = ("Ms0", "beta", "c2", "c4", "c0", "Kq", "K1T", "ax", "ay", "az", "sigma", "me")
        arr = {k: np.zeros(N) for k in names}
        arr["az"][:] = 1.0; arr["beta"][:] = 1.0
        key = reg.astype(np.int64) * (1 << 32) + self.T_cell.astype(np.float32).view(np.uint32).astype(np.int64)
        uniq, inv = np.unique(key, return_inverse=True)
        cls = {k: np.zeros(uniq.size) for k in names}
        first = np.zeros(uniq.size, dtype=np.int64)
        first[inv[::-1]] = np.arange(N - 1, -1, -1)
        for q in range(uniq.size):
            c = first[q]; r = self.regions[reg[c]]; T = self.T_cell[c]
            cls["beta"][q] = 1.0 / (KB * T) if T > 0 else np.nan
            if r.Ms0 <= 0:
                cls["az"][q] = 1.0
                continue
            if not (T > 0):
                raise ValueError("T <= 0")
            th = thermal(T, r.Tc, r.mu_atom, self.V, r.Ms0)
            al = np.sqrt(r.ax ** 2 + r.ay ** 2 + r.az ** 2) or 1.0
            cls["Ms0"][q] = r.Ms0; cls["c2"][q] = th["c2"]; cls["c4"][q] = th["c4"]; cls["c0"][q] = th["c0"]
            cls["Kq"][q] = r.K1 * th["me"]; cls["K1T"][q] = r.K1 * th["me"] ** 3
            cls["ax"][q], cls["ay"][q], cls["az"][q] = r.ax / al, r.ay / al, r.az / al
            cls["sigma"][q] = self.sigma_user if self.sigma_user >= 0 else th["sigma13"]
            cls["me"][q] = th["me"]
        for k in names:
            arr[k] = np.ascontiguousarray(cls[k][inv])
        # cubic anisotropy (Eq. (12); K(T) = K me^(l(l+1)/2), l = 4 and 6)
        self.has_cubic = any(r.Ms0 > 0 and (r.K1c != 0 or r.K2c != 0) for r in self.regions)
        if self.has_cubic:
            k1 = np.zeros(uniq.size); k2 = np.zeros(uniq.size); ax9 = np.zeros((uniq.size, 9))
            for q in range(uniq.size):
                r = self.regions[reg[first[q]]]
                ax9[q] = cubic_axes(r)
                if r.Ms0 > 0:
                    k1[q] = r.K1c * cls["me"][q] ** 10; k2[q] = r.K2c * cls["me"][q] ** 21
            arr["K1cT"] = np.ascontiguousarray(k1[inv]); arr["K2cT"] = np.ascontiguousarray(k2[inv])
            arr["cub"] = np.ascontiguousarray(ax9[inv])
        # 4th-order uniaxial term of Eq. (11): K2(T) = K2 me^10 (l = 4); zero at and above Tc (me = 0)
        self.has_k2 = any(r.Ms0 > 0 and r.K2 != 0 for r in self.regions)
        if self.has_k2:
            k2 = np.array([self.regions[reg[first[q]]].K2 * cls["me"][q] ** 10 for q in range(uniq.size)])
            arr["K2T"] = np.ascontiguousarray(k2[inv])
            arr["me2"] = np.ascontiguousarray(np.where(cls["me"] > 0, cls["me"] ** 2, 1.0)[inv])
        self.coef = arr
        self._dirty = False

    def _problem(self):
        self._setup()
        p = _Problem()
        p.nx, p.ny, p.nz, p.pbc = self.nx, self.ny, self.nz, self.pbc
        p.dx, p.dy, p.dz = self.dx, self.dy, self.dz
        p.active = self.active.ctypes.data
        p.region = self.region_of_cell.ctypes.data
        p.inter_region_exchange = self.inter_region_exchange
        for k in ("Ms0", "beta", "c2", "c4", "c0", "Kq", "K1T", "ax", "ay", "az", "sigma"):
            setattr(p, k, self.coef[k].ctypes.data)
        p.A0, p.D0 = self.A0, self.D0
        p.Bext = (C.c_double * 3)(*self.Bext)
        if self.demag_enabled and self.bd is not None:
            p.bdx, p.bdy, p.bdz = (b.ctypes.data for b in self.bd)
        else:
            p.bdx = p.bdy = p.bdz = None
        p.one_minus_cos_cone = 2.0 * np.sin(0.5 * np.deg2rad(self.cone_deg)) ** 2
        p.seed = self.seed
        if self.has_cubic:
            p.K1cT, p.K2cT, p.cub = (self.coef[k].ctypes.data for k in ("K1cT", "K2cT", "cub"))
        else:
            p.K1cT = p.K2cT = p.cub = None
        if self.has_k2:
            p.K2T, p.me2 = self.coef["K2T"].ctypes.data, self.coef["me2"].ctypes.data
        else:
            p.K2T = p.me2 = None
        return p

    # -- demag ----------------------------------------------------------------------------
    def demag_field(self):
        """B_d (tesla) of the current state, three flat arrays (Eq. (14))."""
        self._setup()
        if self._demag is None:
            self._demag = DemagFFT(self.nx, self.ny, self.nz, self.dx, self.dy, self.dz, self.demag_r_near)
        sh = (self.nz, self.ny, self.nx)
        M = [(self.coef["Ms0"] * a).reshape(sh) for a in self.m]
        return [np.ascontiguousarray(b.ravel()) for b in self._demag.field(*M)]

    # -- iteration --------------------------------------------------------------------------
    def colour_pass(self, colour, dump=False, order=None):
        """One colour pass at the current sweep counter (does not advance it).  With dump=True
        returns dict(dm[N,3], terms[N,6], margin[N], accepted[N])."""
        p = self._problem()
        N = self.N
        d = None
        ptrs = [None] * 4
        if dump:
            d = dict(dm=np.zeros((N, 3)), terms=np.zeros((N, 6)), margin=np.full(N, np.nan), accepted=np.zeros(N, dtype=np.uint8))
            ptrs = [d["dm"].ctypes.data, d["terms"].ctypes.data, d["margin"].ctypes.data, d["accepted"].ctypes.data]
        tri = C.c_int64()
        if order is not None:
            order = np.ascontiguousarray(order, dtype=np.int64)
        acc = lib().orc_colour_pass(C.byref(p), _dp(self.m[0]), _dp(self.m[1]), _dp(self.m[2]), int(colour),
                                    self.sweep, None if order is None else order.ctypes.data,
                                    0 if order is None else order.size, int(self.store_fp32),
                                    *ptrs, C.byref(tri))
        self.accepted += acc; self.trials += tri.value
        self._win_acc += acc; self._win_tri += tri.value
        return d

    def sweep_once(self, dump=False):
        """O6: [demag] -> red -> [demag iff updates_per_sweep == 2] -> black -> counter++; then S11.
        With dump=True returns the per-cell dumps of the two passes (see colour_pass)."""
        if self.demag_enabled:
            self.bd = self.demag_field()
        dumps = [self.colour_pass(0, dump=dump)]
        if self.demag_enabled and self.demag_updates == 2:
            self.bd = self.demag_field()
        dumps.append(self.colour_pass(1, dump=dump))
        self.sweep += 1
        self._win_sweeps += 1
        if self._win_sweeps == 100:
            # PAPER.md:100 + reading G11: every 100 iterations, +-1 deg outside 0.5 +- 0.05, clamp [1, 180]
            if self.adaptive and self._win_tri > 0:
                rate = self._win_acc / self._win_tri
                if rate > 0.55: self.cone_deg = min(180.0, self.cone_deg + 1.0)
                elif rate < 0.45: self.cone_deg = max(1.0, self.cone_deg - 1.0)
            self._win_acc = self._win_tri = self._win_sweeps = 0
        return dumps if dump else None

    def run(self, n_sweeps):
        for _ in range(n_sweeps):
            self.sweep_once()

    def exact_demag_dF(self, cell, dm, b=None):
        """beta dE_demag of the single-cell move dm with the exact field of the current state (+ self term)."""
        p = self._problem()
        if self._demag is None:
            self._demag = DemagFFT(self.nx, self.ny, self.nz, self.dx, self.dy, self.dz, self.demag_r_near)
        tab = np.ascontiguousarray(self._demag.tab)
        b = [np.ascontiguousarray(x, dtype=np.float64) for x in (self.demag_field() if b is None else b)]
        dm = np.ascontiguousarray(dm, dtype=np.float64)
        return lib().orc_exact_demag_dF(C.byref(p), _dp(tab), _dp(b[0]), _dp(b[1]), _dp(b[2]), int(cell), _dp(dm))

    def run_serial_exact(self, n_sweeps):
        """Validation mode (Appendix B): serial MMC, cells one after the other, with the
        exact demag energy change (current field + self term) and the field updated after every accepted move.  The
        oracle's parallel mode is the paper's approximation of this; Appendix B claims no statistical difference."""
        p = self._problem()
        if self._demag is None:
            self._demag = DemagFFT(self.nx, self.ny, self.nz, self.dx, self.dy, self.dz, self.demag_r_near)
        tab = np.ascontiguousarray(self._demag.tab)
        b = [np.ascontiguousarray(x, dtype=np.float64) for x in self.demag_field()]
        for _ in range(n_sweeps):
            tri = C.c_int64()
            acc = lib().orc_serial_exact_sweep(C.byref(p), _dp(self.m[0]), _dp(self.m[1]), _dp(self.m[2]), _dp(tab),
                                               _dp(b[0]), _dp(b[1]), _dp(b[2]), self.sweep, int(self.store_fp32), C.byref(tri))
            self.accepted += acc; self.trials += tri.value
            self.sweep += 1
        self.bd = b
        return b

    def histogram(self, kind, nbins, lo, hi):
        """The paper's verification read-outs over the non-empty cells: kind "length": x = |m|; kind "angle":
        x = polar angle between m and the mean direction, "for each micromagnetic magnetization configuration the mean
        direction is obtained, and for each vector ... the polar angle theta to this mean direction is found".
        Equal bins over [lo, hi): bin = floor((x - lo) nbins / (hi - lo)); returns (counts, under, over)."""
        self._setup()
        act = np.asarray(self.coef["Ms0"]) > 0
        m = np.stack([np.asarray(self.m[a], dtype=np.float64)[act] for a in range(3)])
        L = np.sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2])
        if kind == "length":
            x = L
        else:
            d = m.sum(axis=1); d = d / np.linalg.norm(d)
            x = np.arccos(np.clip((m[0] * d[0] + m[1] * d[1] + m[2] * d[2]) / L, -1.0, 1.0))
        t = (x - lo) * (nbins / (hi - lo))
        under = int(np.count_nonzero(~(t >= 0.0))); over = int(np.count_nonzero(t >= nbins))
        ok = (t >= 0.0) & (t < nbins)
        counts = np.bincount(t[ok].astype(np.int64), minlength=nbins).astype(np.uint64)
        return counts, under, over

    def relax(self, direction, chunk_sweeps=2000, min_chunks=2, max_chunks=50, threshold=0.01):
        """Chunked convergence of one field step: "a chunk with a fixed number of iterations (2000) is
        defined, with an ensemble average magnetization value computed for each chunk ... executed for at least 2 chunks
        ... if their respective final average magnetization values along the applied field direction are close enough
        within an acceptance threshold (0.01 normalized change ...) the computation accepts the last chunk average".
        Reading: the chunk average is the mean over non-empty cells of the state after each iteration,
        averaged over the chunk's iterations; "normalized change" = absolute change of <M_par>/Ms0."""
        u = np.asarray(direction, dtype=np.float64); u = u / np.linalg.norm(u)
        self._setup()
        act = np.asarray(self.coef["Ms0"]) > 0
        prev = 0.0; res = None
        for n in range(1, max_chunks + 1):
            acc = np.zeros(3); acc_len = 0.0
            for _ in range(chunk_sweeps):
                self.sweep_once()
                acc += np.array([self.m[a][act].mean() for a in range(3)])
                acc_len += np.sqrt(self.m[0] ** 2 + self.m[1] ** 2 + self.m[2] ** 2)[act].mean()
            mean = acc / chunk_sweeps
            par = float(mean @ u)
            res = dict(chunks_done=n, converged=False, mean_par_last=par, mean_par_prev=prev, mean_m=mean,
                       mean_len=acc_len / chunk_sweeps, sweeps=n * chunk_sweeps)
            if n >= min_chunks and abs(par - prev) <= threshold:
                res["converged"] = True
                break
            prev = par
        return res

    def colour_terms_given_dm(self, colour, dm):
        """O4 for every active cell of `colour` with caller-supplied trial vectors dm[N,3] -> terms[N,6] (NaN elsewhere)."""
        p = self._problem()
        dm = np.ascontiguousarray(dm, dtype=np.float64)
        t = np.full((self.N, 6), np.nan)
        lib().orc_colour_terms_given_dm(C.byref(p), _dp(self.m[0]), _dp(self.m[1]), _dp(self.m[2]), int(colour), _dp(dm), _dp(t))
        return t

    def cell_dF(self, i, j, k, dm):
        p = self._problem()
        t = np.zeros(6); dm = np.ascontiguousarray(dm, dtype=np.float64)
        lib().orc_cell_dF(C.byref(p), _dp(self.m[0]), _dp(self.m[1]), _dp(self.m[2]), i, j, k, _dp(dm), _dp(t))
        return t

    def observables(self):
        """O8.  Energies in joule; E_demag uses the field of the *current* state."""
        if self.demag_enabled:
            self.bd = self.demag_field()
        p = self._problem()
        E = np.zeros(6); mean = np.zeros(4); na = C.c_int64()
        lib().orc_observables(C.byref(p), _dp(self.m[0]), _dp(self.m[1]), _dp(self.m[2]), _dp(E), _dp(mean), C.byref(na))
        return dict(mean_m=mean[:3].copy(), mean_len=mean[3], E_ex=E[0], E_an=E[1], E_zee=E[2], E_dmi=E[3],
                    E_demag=E[4], E_long=E[5], accepted=self.accepted, trials=self.trials,
                    sweeps_done=self.sweep, cone_deg=self.cone_deg, n_active=na.value)
