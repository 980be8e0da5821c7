"""mmc_mean_m_static (include/mmc.h): the allocation-free read-out of <m>, <|m|> whose scratch is a static device array
of the library, against the existing read-out (mmc_get_observables) on the same state, at the tolerance the other GPU tests
use for these means (test_gpu_parity.py: atol 1e-6 on <m>, rel 1e-6 on <|m|>), on calls in a row that share the array.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _gpu(wl):
    import paper_2106_05593_b200 as P
    s = P.MMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask)
    W.configure(s, wl, P.Material)
    return s


def _agree(out5, ob, wl):
    o = out5.cpu().numpy()
    assert o[4] == wl.n_active, (o[4], wl.n_active)                        # the count is exact
    assert np.allclose(o[:3], ob["mean_m"], atol=1e-6), (o[:3], ob["mean_m"])
    assert o[3] == pytest.approx(ob["mean_len"], rel=1e-6)
    # same per-cell arithmetic on both sides, only the order of the fp64 additions differs
    assert np.abs(o[:3] - ob["mean_m"]).max() < 1e-11 and abs(o[3] - ob["mean_len"]) < 1e-11


def test_static_scratch_readout_matches_the_ctx_readout_on_calls_in_a_row():
    import paper_2106_05593_b200 as P
    big = W.cfg5(nx=384, ny=320)            # 122 880 sites = 30 blocks of 4096, ~30 % magnetic: empty cells must not count
    small = W.cfg4(nx=37, ny=19, nz=3)      # 2109 cells: one ragged block; reads slot 0 of the array the big call filled
    assert 0 < big.n_active < big.N
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    gb, gs = _gpu(big), _gpu(small)
    for it in range(2):                     # big, small, big, small: four calls in a row on one stream, new data each time
        for g, wl in ((gb, big), (gs, small)):
            g.sweep(2)
            ob = g.observables()
            m = g.get_m()
            out.fill_(float("nan"))
            assert P.mean_m_static(m[0], m[1], m[2], out) is out
            torch.cuda.synchronize()
            _agree(out, ob, wl)
    # back to back with no host synchronisation in between: the second call's ticket reset is ordered after the first
    # call's kernel by the stream, and each call wrote the output it was given
    mb, ms = gb.get_m(), gs.get_m()
    o1 = torch.zeros(5, dtype=torch.float64, device="cuda"); o2 = torch.zeros_like(o1); o3 = torch.zeros_like(o1)
    P.mean_m_static(*mb, o1); P.mean_m_static(*ms, o2); P.mean_m_static(*mb, o3)
    torch.cuda.synchronize()
    _agree(o1, gb.observables(), big); _agree(o2, gs.observables(), small)
    assert torch.equal(o1, o3)              # fixed summation order: bit-identical on a repeat
    gb.close(); gs.close()


def test_static_scratch_limits_and_degenerate_sizes():
    import paper_2106_05593_b200 as P
    L = P.lib()
    out = torch.full((5,), 7.0, dtype=torch.float64, device="cuda")
    z = torch.zeros(8, dtype=torch.float32, device="cuda")
    with pytest.raises(P.MMCError) as e:    # refused before anything is enqueued or any buffer is looked at
        P.mean_m_static(z, z, z, out, n_cells=P.STATIC_MAX_CELLS + 1)
    assert e.value.code == P.E_TOO_LARGE and "16777216" in str(e.value)
    torch.cuda.synchronize()
    assert torch.all(out == 7.0)
    assert L.mmc_mean_m_static(None, z.data_ptr(), z.data_ptr(), 8, out.data_ptr(), 0, None) == -1
    assert L.mmc_mean_m_static(z.data_ptr(), z.data_ptr(), z.data_ptr(), -1, out.data_ptr(), 0, None) == -1
    assert L.mmc_mean_m_static(z.data_ptr(), z.data_ptr(), z.data_ptr(), 8, out.data_ptr(), 64, None) == -1
    P.mean_m_static(z, z, z, out)           # no magnetic cell at all: zeros, not NaN
    torch.cuda.synchronize()
    assert torch.all(out == 0.0)
    out.fill_(7.0)
    P.mean_m_static(z, z, z, out, n_cells=0)
    torch.cuda.synchronize()
    assert torch.all(out == 0.0)
    # the largest size it accepts: 4096 blocks, every partial slot of the array in use; closed form of the sums
    n = P.STATIC_MAX_CELLS
    x = torch.full((n,), 0.5, dtype=torch.float32, device="cuda"); y = torch.zeros_like(x); zz = torch.full_like(x, -0.25)
    x[::3] = 0.0; zz[::3] = 0.0             # every third cell empty
    P.mean_m_static(x, y, zz, out)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    n_act = n - (n + 2) // 3
    assert o[4] == n_act and o[0] == 0.5 and o[1] == 0.0 and o[2] == -0.25
    assert o[3] == pytest.approx(float(np.sqrt(np.float32(0.3125))), rel=1e-12)
    # and right after it a one-block call: the 4095 stale partials of the large call are not read
    a = torch.tensor([0.0, 3.0, 0.0, 0.0], dtype=torch.float32, device="cuda"); b = torch.tensor([0.0, 4.0, 0.0, 1.0], dtype=torch.float32, device="cuda")
    c = torch.zeros(4, dtype=torch.float32, device="cuda")
    P.mean_m_static(a, b, c, out)
    torch.cuda.synchronize()
    assert out.cpu().numpy().tolist() == [1.5, 2.5, 0.0, 3.0, 2.0]


def test_static_scratch_call_is_capturable_into_a_cuda_graph():
    """What the entry point is for: issued while its stream is being captured (an allocation would fail the capture), then
    replayed on new data.  The set-up call (symbol look-up) happened outside the capture, as mmc.h asks."""
    import paper_2106_05593_b200 as P
    n = 3 * 4096 + 123
    gen = torch.Generator(device="cuda").manual_seed(5)
    m = [torch.randn(n, dtype=torch.float32, device="cuda", generator=gen) * 0.5 for _ in range(3)]
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    P.mean_m_static(*m, out, n_cells=0)     # set-up outside the capture
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        graph.capture_begin()
        P.mean_m_static(*m, out, stream=s)
        graph.capture_end()
    torch.cuda.synchronize()
    for rep in range(2):
        if rep:
            for t in m:
                t.mul_(0.5).add_(0.125)
        graph.replay()
        torch.cuda.synchronize()
        md = [t.double() for t in m]
        ln = torch.sqrt((md[0] ** 2 + md[1] ** 2 + md[2] ** 2).float()).double()      # fp32 root of the fp64 square sum
        o = out.cpu().numpy()
        assert o[4] == n
        assert np.allclose(o[:3], [float(t.mean()) for t in md], atol=1e-12) and o[3] == pytest.approx(float(ln.mean()), rel=1e-12)
