"""Helpers shared by the GPU parity tests: explain, cell by cell, every difference between the state the CUDA path holds
after one whole iteration (production kernels, no per-cell dump) and the oracle's replay of that iteration.

A cell's trial vector does not depend on its neighbours, so after one iteration every active cell of the CUDA path must
hold either the oracle's accepted candidate fp32(m + dm) or the untouched m: anything else is an arithmetic defect, not a
near-margin decision.  A cell whose decision differs from the oracle's ("flip") must be explained by the oracle's own
numbers: its margin lies inside the window in which fp32 and fp64 may disagree (north_star: 1e-4; plus the carried
stage-1/2 error 2e-6 sum|terms|, plus the demag field tolerance when each side computes its own field), or it is a black
cell next to a red flip (its neighbourhood then differs between the two sides), or -- with a second field update before
the black pass -- a black cell close enough to a red flip for the flip's dipole field to move its margin across zero."""
import numpy as np

MU0 = 4e-7 * np.pi


def explain_iteration(wl, o, m_gpu, field_tol=2e-5, state_tol=2e-6):
    """o: the oracle holding the state BEFORE the iteration (same seed / sweep counter as the CUDA path); m_gpu: the CUDA
    path's state after it (three float64 arrays, natural order).  Runs the oracle's iteration and returns a dict with the
    number of flips, of unexplained flips and of cells holding neither candidate."""
    nx, ny, nz = wl.nx, wl.ny, wl.nz
    N = nx * ny * nz
    m0 = o.get_m()
    d_red, d_black = o.sweep_once(dump=True)
    idx = np.arange(N)
    ci, cj, ck = idx % nx, (idx // nx) % ny, idx // (nx * ny)
    black = ((ci + cj + ck) & 1).astype(bool)
    pick = lambda key: np.where(black if d_red[key].ndim == 1 else black[:, None], d_black[key], d_red[key])
    dm, terms, margin, oacc = pick("dm"), pick("terms"), pick("margin"), pick("accepted").astype(bool)
    act = ~np.isnan(margin)
    near_acc = np.ones(N, bool); near_rej = np.ones(N, bool)
    for a in range(3):
        cand = (m0[a] + dm[:, a]).astype(np.float32).astype(np.float64)
        near_acc &= np.abs(m_gpu[a] - cand) <= state_tol
        near_rej &= np.abs(m_gpu[a] - m0[a]) <= state_tol
    neither = act & ~near_acc & ~near_rej
    flip = act & ~neither & ((oacc & ~near_acc) | (~oacc & ~near_rej))
    untouched_ok = all(np.array_equal(m_gpu[a][~act], m0[a][~act]) for a in range(3))
    # the window of the oracle's margin inside which the two precisions may decide differently
    bzee = o.coef["beta"] * o.V * o.coef["Ms0"]                     # beta V Ms0 per cell (1/tesla)
    dmn = np.linalg.norm(np.where(np.isnan(dm), 0.0, dm), axis=1)
    window = 1e-4 + 2e-6 * np.abs(np.where(np.isnan(terms), 0.0, terms)).sum(axis=1)
    if o.demag_enabled and o.bd is not None and field_tol > 0:
        window = window + bzee * dmn * field_tol * max(np.abs(b).max() for b in o.bd)
    explained = np.abs(np.where(act, margin, np.inf)) < window
    red_flip = flip & ~black
    if red_flip.any():
        # black cells next to a red flip (6-stencil, periodic wrap): exchange and DMI see a different neighbour
        grid = red_flip.reshape(nz, ny, nx)
        nb = np.zeros_like(grid)
        for ax, n, bit in ((2, nx, 1), (1, ny, 2), (0, nz, 4)):
            if n < 2:
                continue
            for sh in (1, -1):
                r = np.roll(grid, sh, axis=ax)
                if not (wl.pbc_mask & bit):
                    sl = [slice(None)] * 3; sl[ax] = 0 if sh == 1 else n - 1
                    r[tuple(sl)] = False
                nb |= r
        explained |= black & nb.ravel()
        if o.demag_enabled and o.demag_updates == 2:
            # second field update: the flip's moment change dM V acts on every black cell as a dipole field,
            # |dB| <= mu0 Ms0 |dm| V / (2 pi r^3): widen the window of the black cells accordingly (flips are few: brute force)
            fl = np.flatnonzero(red_flip)
            pos = np.stack([ci * wl.dx, cj * wl.dy, ck * wl.dz], axis=1)
            extra = np.zeros(N)
            for c in fl:
                r = np.linalg.norm(pos - pos[c], axis=1); r[c] = np.inf
                extra += MU0 * o.coef["Ms0"][c] * dmn[c] * o.V / (2.0 * np.pi * r ** 3)
            explained |= black & (np.abs(np.where(act, margin, np.inf)) < window + bzee * dmn * extra)
    return dict(flips=int(flip.sum()), unexplained=int((flip & ~explained).sum()), neither=int(neither.sum()),
                untouched_ok=bool(untouched_ok), active=int(act.sum()), oracle_accepted=int(oacc[act].sum()),
                flip_cells=np.flatnonzero(flip))
