"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (variant AUTO, default plan).

The oracle cannot step 4096^2 or 16384^2 grids in seconds, so the full-size runs are checked on sampled outputs the
oracle computes exactly: one RK4 step has a domain of dependence of 4 cells (one per stage: N_halo = 4),
so a w x w window of the state after s steps depends only on the (w + 8 s)^2 window of the inputs around it.  The
oracle steps that input window as a small periodic grid; its outer 4 s cells are contaminated by the artificial wrap
and dropped, the inner w x w cells are the exact oracle result of the full-size problem.  Windows sit in the bulk, across
the periodic x edge, and on the wrap corner, i.e. across strip, chunk and wrap seams of the launch plan.
The batched ensemble (cfg5, 512 x 256^2) is small enough per realisation to be compared in full.
Bars as everywhere (BASELINE.json north_star): relative L2 <= 2e-5 (complex fp32), <= 1e-12 (complex fp64); integer
noise words bit-exact."""
import numpy as np
import pytest

import oracle as orc
from paper_2411_18341_b200 import workloads as wl
from helpers import TOL, make_gpu, rel_l2

pytestmark = pytest.mark.gpu

S = 8          # steps
WIN = 64       # window edge
M = 4 * S      # margin the oracle needs around the window


def _idx(start, n):
    return np.arange(start - M, start + WIN + M) % n


def _window_oracle(w, x0, y0):
    """Oracle state after S steps on the window whose inner WIN x WIN cells start at (x0, y0); returns dict of inner windows."""
    ix, iy = _idx(x0, w.nx), _idx(y0, w.ny)
    sel = np.ix_(iy, ix)
    n = WIN + 2 * M
    o = orc.Oracle(n, n, w.dx, w.dy, orc.make_params(**w.params), model=w.model, batch=1, prec32=(w.prec == "c32"),
                   V=None if w.V is None else w.V[sel].astype(np.float64),
                   P=None if w.P is None else w.P[sel].astype(np.float64))
    for name, arr in w.fields.items():
        o.set_field(name, arr[0][sel])
    o.step_rk4(S)
    return {name: getattr(o, name)[0, M:M + WIN, M:M + WIN] for name in w.fields}


def _check_windows(w, corners):
    g = make_gpu(w)                       # variant AUTO, default plan: what bench.py times
    g.step_rk4(S)
    got = {name: g.read_field(name) for name in w.fields}
    variant = g.get_variant()
    g.destroy()
    for (x0, y0) in corners:
        ref = _window_oracle(w, x0, y0)
        ix, iy = np.arange(x0, x0 + WIN) % w.nx, np.arange(y0, y0 + WIN) % w.ny
        for name in w.fields:
            err = rel_l2(got[name][0][np.ix_(iy, ix)], ref[name])
            assert err <= TOL[w.prec], f"{w.name} {name} window ({x0},{y0}) variant {variant}: rel L2 {err:.3e}"


def _corners(n):
    # bulk (crossing a 56- and a 120-column strip seam and a chunk seam), periodic x edge, wrap corner
    return [(n // 2 - 20, n // 2 - 30), (n - WIN // 2, n // 3), (n - WIN // 2, n - WIN // 2)]


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg2_4096_windows(prec):
    w = wl.cfg2(n=4096, prec=prec)
    _check_windows(w, _corners(4096))


def test_cfg3_4096_windows():
    w = wl.cfg3(n=4096, prec="c32")
    _check_windows(w, _corners(4096))


def test_cfg4_16384_windows():
    w = wl.cfg4(n=16384, prec="c32")       # 2 x 2 GiB of state, 16 GiB of workspace planes
    _check_windows(w, _corners(16384))


def test_cfg5_full_ensemble():
    w = wl.cfg5(n=256, batch=512, prec="c32")
    g = make_gpu(w)
    # integer noise stream of every cell of every realisation, first, second and last step of the 20 000
    for step in (0, 1, 19999):
        assert np.array_equal(g.debug_noise_u32(step), orc.noise_u32(256, 256, 512, w.seed, step)), f"step {step}"
    n_steps = 3
    g.step_rk4(n_steps)
    o = orc.Oracle(w.nx, w.ny, w.dx, w.dy, orc.make_params(**w.params), model=w.model, batch=w.batch, prec32=True,
                   noise=True, seed=w.seed, P=w.P.astype(np.float64))
    for name, arr in w.fields.items():
        o.set_field(name, arr)
    o.step_rk4(n_steps)
    for name in w.fields:
        got = g.read_field(name)
        ref = getattr(o, name)
        for r in range(w.batch):
            err = rel_l2(got[r], ref[r])
            assert err <= TOL["c32"], f"realisation {r} {name}: rel L2 {err:.3e}"
    mean = g.ensemble_mean_density("psi_p")
    assert rel_l2(mean, o.ensemble_mean_density("psi_p")) <= TOL["c32"]
    g.destroy()


# ---- late segments: the oracle restarted from a GPU checkpoint far into the run (SURVEY.md 8(c) "horizons") ----------
def _check_windows_from_checkpoint(w, n_before, corners):
    """Steps the GPU n_before steps, checkpoints, steps S more; the oracle redoes the S steps from the checkpoint."""
    import dataclasses
    g = make_gpu(w)
    g.step_rk4(n_before)
    snap = {name: g.read_field(name) for name in w.fields}
    for name, arr in snap.items():
        assert np.all(np.isfinite(arr)), name
    g.step_rk4(S)
    got = {name: g.read_field(name) for name in w.fields}
    g.destroy()
    w2 = dataclasses.replace(w, fields=snap)
    for (x0, y0) in corners:
        ref = _window_oracle(w2, x0, y0)
        ix, iy = np.arange(x0, x0 + WIN) % w.nx, np.arange(y0, y0 + WIN) % w.ny
        for name in w.fields:
            err = rel_l2(got[name][0][np.ix_(iy, ix)], ref[name])
            assert err <= TOL[w.prec], f"{w.name} {name} window ({x0},{y0}) after {n_before} steps: rel L2 {err:.3e}"


def test_cfg2_4096_segment_at_step_5000():
    _check_windows_from_checkpoint(wl.cfg2(n=4096, prec="c32"), 5000, _corners(4096))


def test_cfg3_4096_segment_at_step_10000():
    # the pumped reservoir has built up and the condensate has grown by then (n0 = 0, psi0 = noise at the start)
    _check_windows_from_checkpoint(wl.cfg3(n=4096, prec="c32"), 10000, _corners(4096))


def test_cfg5_last_steps_of_the_run():
    w = wl.cfg5(n=256, batch=512, prec="c32")
    n_before, n_last = w.n_steps - 2, 2          # steps 19 998 and 19 999 of the 20 000
    g = make_gpu(w)
    g.step_rk4(n_before)
    snap = {name: g.read_field(name) for name in w.fields}
    g.step_rk4(n_last)
    assert g.get_step() == w.n_steps
    o = orc.Oracle(w.nx, w.ny, w.dx, w.dy, orc.make_params(**w.params), model=w.model, batch=w.batch, prec32=True,
                   noise=True, seed=w.seed, P=w.P.astype(np.float64))
    for name, arr in snap.items():
        assert np.all(np.isfinite(arr)), name
        o.set_field(name, arr)
    o.step = n_before                            # the step index keys the noise
    o.step_rk4(n_last)
    for name in w.fields:
        got, ref = g.read_field(name), getattr(o, name)
        worst = max(rel_l2(got[r], ref[r]) for r in range(w.batch))
        assert worst <= TOL["c32"], f"{name}: worst realisation rel L2 {worst:.3e}"
    g.destroy()
