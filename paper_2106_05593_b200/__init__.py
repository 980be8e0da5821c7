"""Thin Python binding of include/mmc.h (argument marshalling only -- every step of the MMC path runs in the
CUDA library ``libmmc_b200.so``).  PyTorch is used for device memory and the stream, nothing else.

There is no CPU fallback: if the shared library is missing or cannot be loaded, importing ``MMC`` users fail
loudly (``MMCLibraryError``); build it with ``python -m paper_2106_05593_b200.build`` or ``__graft_entry__.build()``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmmc_b200.so")

MUB = 9.2740100783e-24

# every symbol include/mmc.h declares
SYMBOLS = [
    "mmc_create", "mmc_destroy", "mmc_set_material", "mmc_set_exchange_coupling", "mmc_set_temperature",
    "mmc_set_field", "mmc_set_move", "mmc_set_demag", "mmc_set_seed", "mmc_set_sweep_counter", "mmc_set_m",
    "mmc_get_m", "mmc_set_m_host", "mmc_get_m_host", "mmc_sweep", "mmc_sweep_timed", "mmc_demag_field", "mmc_get_observables", "mmc_reset_counters", "mmc_reset_averages", "mmc_relax", "mmc_histogram",
    "mmc_debug_pass", "mmc_thermal", "mmc_demag_tensor_at", "mmc_mean_m_static", "mmc_strerror", "mmc_last_error",
]

STATIC_MAX_CELLS = 1 << 24          # MMC_STATIC_MAX_CELLS of include/mmc.h
E_TOO_LARGE = -7                    # MMC_E_TOO_LARGE


class MMCLibraryError(RuntimeError):
    pass


class MMCError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mmc error {code}: {msg}")
        self.code = code


class Material(C.Structure):
    """mmc_material (SI units; Ms0 == 0 marks an empty region)."""
    _fields_ = [(n, C.c_double) for n in ("Ms0", "A0", "K1", "ax", "ay", "az", "D0", "Tc", "mu_atom",
                                          "K1c", "K2c", "c1x", "c1y", "c1z", "c2x", "c2y", "c2z", "K2")]

    def __init__(self, Ms0=0.0, A0=0.0, K1=0.0, ax=0.0, ay=0.0, az=1.0, D0=0.0, Tc=1.0, mu_atom=MUB,
                 K1c=0.0, K2c=0.0, c1x=1.0, c1y=0.0, c1z=0.0, c2x=0.0, c2y=1.0, c2z=0.0, K2=0.0):
        super().__init__(Ms0, A0, K1, ax, ay, az, D0, Tc, mu_atom, K1c, K2c, c1x, c1y, c1z, c2x, c2y, c2z, K2)


class Obs(C.Structure):
    """mmc_obs."""
    _fields_ = [("mean_m", C.c_double * 3), ("mean_len", C.c_double),
                ("E_ex", C.c_double), ("E_an", C.c_double), ("E_zee", C.c_double), ("E_dmi", C.c_double),
                ("E_demag", C.c_double), ("E_long", C.c_double),
                ("accepted", C.c_uint64), ("trials", C.c_uint64), ("sweeps_done", C.c_uint64),
                ("cone_deg", C.c_double), ("sigma_used", C.c_double),
                ("run_mean_m", C.c_double * 3), ("run_mean_len", C.c_double), ("run_sweeps", C.c_uint64)]


class RelaxResult(C.Structure):
    """mmc_relax_result."""
    _fields_ = [("chunks_done", C.c_int), ("converged", C.c_int), ("mean_par_last", C.c_double), ("mean_par_prev", C.c_double),
                ("mean_m", C.c_double * 3), ("mean_len", C.c_double), ("sweeps", C.c_uint64)]


_lib = None


def lib():
    """Load libmmc_b200.so and declare the prototypes of include/mmc.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MMCLibraryError(f"{LIB_PATH} not built: run `python -m paper_2106_05593_b200.build` (no CPU fallback exists)")
    try:
        L = C.CDLL(LIB_PATH)
    except OSError as e:  # pragma: no cover
        raise MMCLibraryError(f"cannot load {LIB_PATH}: {e}") from e
    vp, i32, u64, dbl = C.c_void_p, C.c_int, C.c_uint64, C.c_double
    L.mmc_create.argtypes = [C.POINTER(vp), i32, i32, i32, dbl, dbl, dbl, C.c_uint, i32, vp]
    L.mmc_destroy.argtypes = [vp]
    L.mmc_set_material.argtypes = [vp, i32, C.POINTER(Material), vp]
    L.mmc_set_exchange_coupling.argtypes = [vp, i32]
    L.mmc_set_temperature.argtypes = [vp, dbl, vp]
    L.mmc_set_field.argtypes = [vp, dbl, dbl, dbl]
    L.mmc_set_move.argtypes = [vp, dbl, dbl, i32]
    L.mmc_set_demag.argtypes = [vp, i32, i32]
    L.mmc_set_seed.argtypes = [vp, u64]
    L.mmc_set_sweep_counter.argtypes = [vp, u64]
    L.mmc_set_m.argtypes = [vp, vp, vp, vp]
    L.mmc_get_m.argtypes = [vp, vp, vp, vp]
    L.mmc_set_m_host.argtypes = [vp, vp, vp, vp]
    L.mmc_get_m_host.argtypes = [vp, vp, vp, vp]
    L.mmc_sweep.argtypes = [vp, i32]
    L.mmc_sweep_timed.argtypes = [vp, i32, C.POINTER(dbl)]
    L.mmc_demag_field.argtypes = [vp, vp, vp, vp]
    L.mmc_get_observables.argtypes = [vp, C.POINTER(Obs)]
    L.mmc_reset_counters.argtypes = [vp]
    L.mmc_reset_averages.argtypes = [vp]
    L.mmc_histogram.argtypes = [vp, i32, i32, dbl, dbl, vp, vp]
    L.mmc_relax.argtypes = [vp, dbl, dbl, dbl, i32, i32, i32, dbl, C.POINTER(RelaxResult)]
    L.mmc_debug_pass.argtypes = [vp, i32, vp, vp, vp, vp]
    L.mmc_thermal.argtypes = [dbl] * 5 + [C.POINTER(dbl)]
    L.mmc_demag_tensor_at.argtypes = [dbl, dbl, dbl, i32, i32, i32, C.POINTER(dbl)]
    L.mmc_mean_m_static.argtypes = [vp, vp, vp, C.c_longlong, vp, i32, vp]
    L.mmc_strerror.argtypes = [i32]; L.mmc_strerror.restype = C.c_char_p
    L.mmc_last_error.argtypes = [vp]; L.mmc_last_error.restype = C.c_char_p
    for s in SYMBOLS:
        if s not in ("mmc_strerror", "mmc_last_error"):
            getattr(L, s).restype = C.c_int
    _lib = L
    return L


def thermal(T, Tc, mu_atom, V, Ms0):
    """Host-side set-up values of the library: dict(me, chi, c2, c4, sigma13, mu2)."""
    o = (C.c_double * 6)()
    rc = lib().mmc_thermal(T, Tc, mu_atom, V, Ms0, o)
    if rc:
        raise MMCError(rc, lib().mmc_strerror(rc).decode())
    return dict(me=o[0], chi=o[1], c2=o[2], c4=o[3], sigma13=o[4], mu2=o[5])


def demag_tensor_at(dx, dy, dz, ox, oy, oz):
    o = (C.c_double * 6)()
    rc = lib().mmc_demag_tensor_at(dx, dy, dz, ox, oy, oz, o)
    if rc:
        raise MMCError(rc, lib().mmc_strerror(rc).decode())
    return np.array(list(o))


def mean_m_static(mx, my, mz, out5, n_cells=None, stream=None):
    """mmc_mean_m_static: enqueue <m>, <|m|> and the number of non-empty cells of the device float32 tensors mx, my, mz into
    the device float64 tensor out5 (5 elements) on `stream` (default: torch's current stream of that device).  The library
    allocates nothing (its scratch is a static device array shared by all calls: do not overlap two of them on the GPU);
    neither does this wrapper: every buffer is the caller's.  Returns out5 (valid after the stream has run)."""
    import torch
    n = int(mx.numel() if n_cells is None else n_cells)
    if n <= STATIC_MAX_CELLS:                      # beyond it the library refuses before it looks at the buffers
        for t in (mx, my, mz):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() >= n and t.device == mx.device
        assert out5.is_cuda and out5.dtype == torch.float64 and out5.is_contiguous() and out5.numel() >= 5 and out5.device == mx.device
    st = stream if stream is not None else torch.cuda.current_stream(mx.device)
    rc = lib().mmc_mean_m_static(mx.data_ptr(), my.data_ptr(), mz.data_ptr(), n, out5.data_ptr(), mx.device.index or 0,
                                 C.c_void_p(st.cuda_stream))
    if rc:
        raise MMCError(rc, lib().mmc_strerror(rc).decode())
    return out5


class MMC:
    """One mmc_ctx.  Method names mirror include/mmc.h; tensors are torch CUDA float32 in natural cell order."""

    def __init__(self, nx, ny, nz, dx, dy, dz, pbc_mask=0, device=0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise MMCLibraryError("a CUDA device is required (no CPU fallback exists)")
        self._torch = torch
        self.nx, self.ny, self.nz = nx, ny, nz
        self.N = nx * ny * nz
        self.device = torch.device("cuda", device)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        L = lib()
        rc = L.mmc_create(C.byref(self._h), nx, ny, nz, dx, dy, dz, pbc_mask, device, C.c_void_p(self._stream.cuda_stream))
        if rc:
            raise MMCError(rc, L.mmc_strerror(rc).decode())

    def _ck(self, rc):
        if rc:
            raise MMCError(rc, lib().mmc_last_error(self._h).decode() or lib().mmc_strerror(rc).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().mmc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- setters --------------------------------------------------------------------------------
    def set_material(self, regions, region_of_cell=None):
        arr = (Material * len(regions))(*regions)
        roc = None
        if region_of_cell is not None:
            roc = np.ascontiguousarray(region_of_cell, dtype=np.int32).ravel()
            assert roc.size == self.N
        self._ck(lib().mmc_set_material(self._h, len(regions), arr, None if roc is None else roc.ctypes.data))

    def set_exchange_coupling(self, inter_region_exchange):
        self._ck(lib().mmc_set_exchange_coupling(self._h, int(inter_region_exchange)))

    def set_temperature(self, T_uniform, T_per_cell=None):
        t = None
        if T_per_cell is not None:
            t = np.ascontiguousarray(T_per_cell, dtype=np.float32).ravel()
            assert t.size == self.N
        self._ck(lib().mmc_set_temperature(self._h, float(T_uniform), None if t is None else t.ctypes.data))

    def set_field(self, Bx, By, Bz):
        self._ck(lib().mmc_set_field(self._h, float(Bx), float(By), float(Bz)))

    def set_move(self, cone_deg, sigma=-1.0, adaptive_cone=False):
        self._ck(lib().mmc_set_move(self._h, float(cone_deg), float(sigma), int(bool(adaptive_cone))))

    def set_demag(self, enabled, updates_per_sweep=1):
        self._ck(lib().mmc_set_demag(self._h, int(bool(enabled)), int(updates_per_sweep)))

    def set_seed(self, seed):
        self._ck(lib().mmc_set_seed(self._h, int(seed)))

    def set_sweep_counter(self, sweep):
        self._ck(lib().mmc_set_sweep_counter(self._h, int(sweep)))

    def _dev(self, a):
        torch = self._torch
        if not isinstance(a, torch.Tensor):
            a = torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32))
        return a.to(device=self.device, dtype=torch.float32).contiguous().view(-1)

    def set_m(self, mx, my, mz):
        t = [self._dev(a) for a in (mx, my, mz)]
        assert all(x.numel() == self.N for x in t)
        self._ck(lib().mmc_set_m(self._h, t[0].data_ptr(), t[1].data_ptr(), t[2].data_ptr()))

    def set_m_device_ptrs(self, px, py, pz):
        self._ck(lib().mmc_set_m(self._h, px, py, pz))

    def set_m_host(self, mx, my, mz):
        """mmc_set_m_host: host tensors / arrays (float32, N each; pinned tensors copy asynchronously)."""
        self._ck(lib().mmc_set_m_host(self._h, *[self._host_ptr(a) for a in (mx, my, mz)]))

    def get_m_host(self, mx, my, mz):
        """mmc_get_m_host: enqueue the copy of m into the given host buffers (valid after a synchronising call)."""
        self._ck(lib().mmc_get_m_host(self._h, *[self._host_ptr(a) for a in (mx, my, mz)]))

    def _host_ptr(self, a):
        if hasattr(a, "data_ptr"):
            assert (not a.is_cuda) and a.dtype == self._torch.float32 and a.is_contiguous() and a.numel() == self.N
            return a.data_ptr()
        assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"] and a.size == self.N
        return a.ctypes.data

    # -- work -----------------------------------------------------------------------------------
    def get_m(self):
        torch = self._torch
        out = [torch.empty(self.N, dtype=torch.float32, device=self.device) for _ in range(3)]
        self._ck(lib().mmc_get_m(self._h, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr()))
        return out

    def sweep(self, n_sweeps=1):
        self._ck(lib().mmc_sweep(self._h, int(n_sweeps)))

    run = sweep

    PHASES = ("pack", "rows_fwd", "columns", "rows_inv", "z_inverse", "red", "black", "end_sweep")

    def sweep_timed(self, n_sweeps=1):
        """mmc_sweep_timed: dict phase -> summed device milliseconds over the n iterations (synchronises)."""
        ms = (C.c_double * 8)()
        self._ck(lib().mmc_sweep_timed(self._h, int(n_sweeps), ms))
        return dict(zip(self.PHASES, list(ms)))

    def demag_field(self, want=True):
        torch = self._torch
        if not want:
            self._ck(lib().mmc_demag_field(self._h, None, None, None))
            return None
        out = [torch.empty(self.N, dtype=torch.float32, device=self.device) for _ in range(3)]
        self._ck(lib().mmc_demag_field(self._h, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr()))
        return out

    def observables(self):
        o = Obs()
        self._ck(lib().mmc_get_observables(self._h, C.byref(o)))
        d = {k: getattr(o, k) for k in ("mean_len", "E_ex", "E_an", "E_zee", "E_dmi", "E_demag", "E_long", "accepted",
                                        "trials", "sweeps_done", "cone_deg", "sigma_used", "run_mean_len", "run_sweeps")}
        d["mean_m"] = np.array(list(o.mean_m)); d["run_mean_m"] = np.array(list(o.run_mean_m))
        return d

    def histogram(self, kind, nbins, lo, hi):
        """mmc_histogram: kind "length" (|m|) or "angle" (polar angle to the mean direction);
        returns (counts uint64[nbins], under, over)."""
        k = {"length": 0, "angle": 1}[kind]
        counts = np.zeros(int(nbins), dtype=np.uint64); uo = np.zeros(2, dtype=np.uint64)
        self._ck(lib().mmc_histogram(self._h, k, int(nbins), float(lo), float(hi), counts.ctypes.data, uo.ctypes.data))
        return counts, int(uo[0]), int(uo[1])

    def relax(self, direction, chunk_sweeps=2000, min_chunks=2, max_chunks=50, threshold=0.01):
        """mmc_relax: chunked convergence of one field step; returns a dict of mmc_relax_result."""
        r = RelaxResult()
        self._ck(lib().mmc_relax(self._h, float(direction[0]), float(direction[1]), float(direction[2]), int(chunk_sweeps),
                                 int(min_chunks), int(max_chunks), float(threshold), C.byref(r)))
        return dict(chunks_done=r.chunks_done, converged=bool(r.converged), mean_par_last=r.mean_par_last,
                    mean_par_prev=r.mean_par_prev, mean_m=np.array(list(r.mean_m)), mean_len=r.mean_len, sweeps=r.sweeps)

    def reset_counters(self):
        self._ck(lib().mmc_reset_counters(self._h))

    def reset_averages(self):
        self._ck(lib().mmc_reset_averages(self._h))

    def debug_pass(self, colour):
        """One colour pass with the per-cell dump: dict(dm[N,3], terms[N,6], margin[N], accepted[N]) (torch, device).
        Untouched entries (other colour, empty cells) hold NaN / 255."""
        torch = self._torch
        dm = torch.full((self.N, 3), float("nan"), dtype=torch.float32, device=self.device)
        terms = torch.full((self.N, 6), float("nan"), dtype=torch.float32, device=self.device)
        margin = torch.full((self.N,), float("nan"), dtype=torch.float32, device=self.device)
        acc = torch.full((self.N,), 255, dtype=torch.uint8, device=self.device)
        self._ck(lib().mmc_debug_pass(self._h, int(colour), dm.data_ptr(), terms.data_ptr(), margin.data_ptr(), acc.data_ptr()))
        return dict(dm=dm, terms=terms, margin=margin, accepted=acc)
