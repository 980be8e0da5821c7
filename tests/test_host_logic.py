"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol include/mmc.h
declares, its fp64 set-up arithmetic (thermal coefficients, demag tensor) agrees with the independently written
oracle, and the N>1 replica sharding works under gloo with world_size 2.  No compute call needs a GPU here."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    from paper_2106_05593_b200 import build as B
    B.build()
    import paper_2106_05593_b200 as P
    return P


def test_library_exports_every_declared_symbol(P):
    with open(os.path.join(ROOT, "include", "mmc.h")) as f:
        hdr = f.read()
    declared = set(re.findall(r"\b(mmc_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(P.SYMBOLS)
    L = P.lib()
    for s in declared:
        assert hasattr(L, s), s
    assert P.lib().mmc_strerror(-2) == b"zero-length magnetisation in a non-empty cell"
    assert P.lib().mmc_last_error(None) == b"null context"


def test_no_gpu_means_loud_failure(P):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(P.MMCLibraryError):
        P.MMC(8, 8, 1, 5e-9, 5e-9, 5e-9)


def test_product_does_not_import_the_oracle():
    """Product and oracle are independent: no file of the package names the oracle package or its library in code, the
    binding never imports it, and the oracle never names the package."""
    pkg = os.path.join(ROOT, "paper_2106_05593_b200")
    pat = re.compile(r"import\s+oracle|from\s+oracle|oracle\.|libmmc_oracle|mmc_oracle\.c|orc_[a-z_0-9]+\s*\(|[\"'/]oracle[\"'/]")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                hits = pat.findall(src)
                assert not hits, (fn, hits)
    for fn in ("include/mmc.h",):
        assert not pat.findall(open(os.path.join(ROOT, fn)).read()), fn
    opat = re.compile(r"(?:import|from)\s+paper_2106_05593_b200|libmmc_b200|#\s*include\s*[\"<][^\">]*mmc(?:_internal)?\.h")
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            assert not opat.findall(open(os.path.join(ROOT, "oracle", fn)).read()), fn
    wsrc = open(os.path.join(ROOT, "workloads", "__init__.py")).read()          # the shared input generators import neither
    assert not re.findall(r"^\s*(?:import|from)\s+(?:oracle|paper_2106_05593_b200)", wsrc, flags=re.M)


def test_explain_iteration_classifies_flips():
    """tests/parity_util.py on the oracle alone: an exact replay has no flips; a decision forced the other way in a cell
    whose margin is far from zero is reported as unexplained; a state that is neither candidate is reported as such."""
    import oracle as O
    import workloads as W
    from parity_util import explain_iteration
    wl = W.cfg2(nx=20, ny=14); wl.adaptive_cone = False

    def orc():
        s = O.OracleMMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, store_fp32=True)
        W.configure(s, wl, O.Material)
        return s
    a = orc(); a.run(1)
    r = explain_iteration(wl, orc(), a.get_m())
    assert r["flips"] == 0 and r["neither"] == 0 and r["unexplained"] == 0 and r["active"] == wl.N and r["untouched_ok"]
    b = orc(); d_red, _ = b.sweep_once(dump=True)
    red = np.flatnonzero(~np.isnan(d_red["margin"]))
    c = red[np.argmax(np.abs(d_red["margin"][red]))]                 # the red cell furthest from the decision boundary
    m = a.get_m()
    m0 = orc().get_m()
    for q in range(3):                                               # force the other decision there
        m[q][c] = m0[q][c] if d_red["accepted"][c] else np.float32(m0[q][c] + d_red["dm"][c, q])
    r = explain_iteration(wl, orc(), m)
    assert r["flips"] >= 1 and r["unexplained"] >= 1 and c in r["flip_cells"]
    m = a.get_m(); m[0][c] += 1e-3
    assert explain_iteration(wl, orc(), m)["neither"] == 1


def test_thermal_setup_matches_oracle(P):
    import oracle as O
    for T, Tc, V, Ms0 in ((300, 870, 1.25e-25, 8e5), (679, 680, 1.25e-25, 8e5), (700, 680, 1.25e-25, 8e5), (680, 680, 1.25e-25, 8e5),
                          (650, 700, 8e-27, 6e5), (699.99, 700, 8e-27, 6e5), (200, 700, 8e-27, 6e5), (500, 870, 2.5e-25, 8.6e5),
                          (300, 655.3, 2.7e-26, 1.1e6), (749.9, 712.0, 2.7e-26, 1.1e6)):
        a = P.thermal(T, Tc, P.MUB, V, Ms0); b = O.thermal(T, Tc, O.MUB, V, Ms0)
        for k in ("me", "c2", "c4", "sigma13"):
            assert a[k] == pytest.approx(b[k], rel=2e-10, abs=1e-300), (T, Tc, k)
        if b["c4"] > 0:
            assert a["mu2"] == pytest.approx(-b["c2"] / (2 * b["c4"]), rel=2e-10, abs=1e-15)
    o = (P.C.c_double * 6)()
    assert P.lib().mmc_thermal(-5.0, 700.0, P.MUB, 1e-26, 8e5, o) == -1


def test_demag_tensor_matches_oracle(P):
    """Library: lattice + second differences in binary128 / moment expansion.  Oracle: 27-point sum / sub-cube dipoles."""
    import oracle as O
    for d in ((1.0, 1.0, 1.0), (5e-9, 5e-9, 10e-9), (2e-9, 3e-9, 4e-9)):
        for o in ((0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (3, 2, 1), (-3, 2, -1), (10, -7, 0), (40, 0, 0), (2, 40, 1)):
            a = P.demag_tensor_at(*d, *o); b = O.newell(o[0] * d[0], o[1] * d[1], o[2] * d[2], *d)
            assert np.allclose(a, b, rtol=1e-12, atol=1e-15 * np.abs(b).max() + 1e-30), (d, o)
        for o in ((41, 0, 0), (41, 30, 2), (100, 60, 0), (45, -45, 3), (0, 0, 41), (300, 200, 0)):
            a = P.demag_tensor_at(*d, *o); b = O.newell(o[0] * d[0], o[1] * d[1], o[2] * d[2], *d)
            assert np.abs(a - b).max() <= 2e-6 * np.abs(b).max(), (d, o)


def test_replica_sharding_gloo_world_size_2():
    """Multi-GPU = replicas only: each rank runs an independent replica with its own seed and the
    aggregate metric is the sum over ranks / max time.  Covers bench.py's rank plumbing with gloo on CPU."""
    code = r'''
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
r, w = dist.get_rank(), dist.get_world_size()
seeds = bench.replica_seed(1234, r)
val = bench.aggregate_over_ranks(units=1000.0 * (r + 1), seconds=0.5 * (r + 1), backend_device="cpu")
if r == 0:
    print(json.dumps({"world": w, "seed0": bench.replica_seed(1234, 0), "seed1": bench.replica_seed(1234, 1), "value": val}))
dist.destroy_process_group()
''' % ROOT
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29533", "-c", code] if False else
                       [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29533", "--no-python", sys.executable, "-c", code],
                       capture_output=True, text=True, env=env, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1]
    out = json.loads(line)
    assert out["world"] == 2 and out["seed0"] != out["seed1"]
    assert out["value"] == pytest.approx((1000.0 + 2000.0) / 1.0)     # total units / max time over ranks


def test_bench_traffic_is_measured_or_null(monkeypatch):
    """bench.py's roofline.traffic: parsed from the committed ncu capture profiles/traffic_cfg<N>.csv only while the sources
    are the ones the capture was taken from (profiles/traffic_cfg<N>.md carries their hash); null after any change."""
    sys.path.insert(0, ROOT)
    import bench
    md = open(os.path.join(ROOT, "profiles", "traffic_cfg4.md")).read()
    recorded = re.search(r"source_hash: ([0-9a-f]{16})", md).group(1)
    monkeypatch.setattr(bench, "source_hash", lambda: recorded)
    t = bench.ncu_traffic(4)
    assert {"colour_pass_kernel", "demag_rows_fwd_kernel", "demag_columns_kernel", "demag_rows_inv_kernel"} <= set(t)
    for k, v in t.items():
        assert v["dram_bytes"] > 1e6 and v["warp_instructions"] > 1e5, k
    # the columns kernel moves about what the algorithm needs (U + T + tensor = 478.6 MB for cfg 4), not multiples of it
    assert 0.5 < t["demag_columns_kernel"]["dram_bytes"] / 478.6e6 < 1.5
    monkeypatch.setattr(bench, "source_hash", lambda: "0" * 16)
    assert bench.ncu_traffic(4) == {}
    assert bench.ncu_traffic(3) == {}            # no capture committed for this config
    assert re.fullmatch(r"[0-9a-f]{16}", __import__("importlib").reload(bench).source_hash())


def test_bench_demag_byte_model():
    """Algorithmic bytes of the demag kernels as DESIGN.md section 6 states them (cfg 4: U 100.8 MB, T 176.3 MB, tensor 201.5 MB)."""
    sys.path.insert(0, ROOT)
    import bench

    class WL:
        nx, ny, nz, N = 1024, 1024, 4, 1024 * 1024 * 4
    b = bench.demag_kernel_bytes(WL, False)
    assert b["columns"]["bytes"] == pytest.approx(478.6e6, rel=2e-3) and b["z_inverse"]["bytes"] == pytest.approx(277.1e6, rel=2e-3)
    assert b["rows_fwd"]["bytes"] == pytest.approx(151.1e6, rel=2e-3) and b["rows_inv"]["bytes"] == b["rows_fwd"]["bytes"]
    WL.nx = WL.ny = 2048; WL.nz = 1; WL.N = 2048 * 2048
    b = bench.demag_kernel_bytes(WL, True)
    assert "z_inverse" not in b and sum(v["bytes"] for v in b.values()) / WL.N == pytest.approx(156, abs=2)


def test_every_environment_knob_is_documented():
    """Every MMC_* environment variable the library reads is named in include/mmc.h and in README.md."""
    import glob
    names = set()
    for f in glob.glob(os.path.join(ROOT, "paper_2106_05593_b200", "csrc", "*")):
        names |= set(re.findall(r'getenv\("(MMC_[A-Z0-9_]+)"\)', open(f).read()))
    assert len(names) >= 8
    hdr = open(os.path.join(ROOT, "include", "mmc.h")).read()
    readme = open(os.path.join(ROOT, "README.md")).read()
    for n in sorted(names):
        assert n in hdr, f"{n} is not documented in include/mmc.h"
        assert n in readme, f"{n} is not named in README.md"
