"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (variant AUTO, default plan),
at the horizons of SURVEY.md section 8(c).

The oracle cannot step 4096^2 or 16384^2 grids for thousands of steps, so the full-size runs are checked
  (1) on the full grid for 20 steps from t = 0 (cfg2 4096^2, both precisions: 35 s of oracle time each), and
  (2) on sampled outputs the oracle computes exactly: one RK4 step has a domain of dependence of 4 cells (one per stage,
      PAPER.md:183: N_halo = 4), so a w x w window of the state after s steps depends only on the (w + 8 s)^2 window of
      the inputs around it.  The oracle steps that input window as a small periodic grid; its outer 4 s cells are
      contaminated by the artificial wrap and dropped, the inner w x w cells are the exact oracle result of the full-size
      problem.  Windows sit in the bulk, on a face (across the periodic x edge) and on the wrap corner, i.e. across strip,
      chunk and wrap seams of the launch plan.
  (3) Late in a run ("segments"): the GPU is stepped n_before steps, checkpointed, stepped s more; the oracle redoes the s
      steps from the checkpoint (windows).  The fp32 error of a full-length run against an fp64 oracle exceeds 2e-5 for
      ANY implementation (1.1e-8 per step), so a run is gated segment by segment.
The batched ensemble (cfg5, 512 x 256^2) is small enough per realisation to be compared in full.
Bars as everywhere (BASELINE.json north_star): relative L2 <= 2e-5 (complex fp32), <= 1e-12 (complex fp64), plus the
element-wise guard of helpers.check_close; integer noise words bit-exact."""
import dataclasses

import numpy as np
import pytest

import oracle as orc
from paper_2411_18341_b200 import workloads as wl
from helpers import TOL, check_close, make_gpu, make_oracle
from test_gpu_horizons import _report

pytestmark = pytest.mark.gpu


def _window_oracle(w, x0, y0, win, steps, step0=0):
    """Oracle state after `steps` steps on the window whose inner win x win cells start at (x0, y0)."""
    m = 4 * steps                               # margin the oracle needs around the window
    ix = np.arange(x0 - m, x0 + win + m) % w.nx
    iy = np.arange(y0 - m, y0 + win + m) % w.ny
    sel = np.ix_(iy, ix)
    n = win + 2 * m
    o = orc.Oracle(n, n, w.dx, w.dy, orc.make_params(**w.params), model=w.model, batch=1, prec32=(w.prec == "c32"),
                   V=None if w.V is None else w.V[sel].astype(np.float64),
                   P=None if w.P is None else w.P[sel].astype(np.float64))
    for name, arr in w.fields.items():
        o.set_field(name, arr[0][sel])
    o.step = step0
    o.step_rk4(steps)
    return {name: getattr(o, name)[0, m:m + win, m:m + win] for name in w.fields}


def _compare_windows(w, got, corners, win, steps, what):
    for (x0, y0) in corners:
        ref = _window_oracle(w, x0, y0, win, steps)
        ix, iy = np.arange(x0, x0 + win) % w.nx, np.arange(y0, y0 + win) % w.ny
        for name in w.fields:
            check_close(got[name][0][np.ix_(iy, ix)], ref[name], TOL[w.prec], f"{w.name} {name} window ({x0},{y0}) {what}")


def _check_windows(w, corners, win, steps):
    g = make_gpu(w)                       # variant AUTO, default plan: what bench.py times
    g.step_rk4(steps)
    got = {name: g.read_field(name) for name in w.fields}
    variant = g.get_variant()
    g.destroy()
    _compare_windows(w, got, corners, win, steps, f"variant {variant}")


def _check_windows_from_checkpoint(w, n_before, corners, win, steps):
    """Steps the GPU n_before steps, checkpoints, steps `steps` more; the oracle redoes them from the checkpoint."""
    g = make_gpu(w)
    g.step_rk4(n_before)
    snap = {name: g.read_field(name) for name in w.fields}
    for name, arr in snap.items():
        assert np.all(np.isfinite(arr)), name
    g.step_rk4(steps)
    got = {name: g.read_field(name) for name in w.fields}
    g.destroy()
    _compare_windows(dataclasses.replace(w, fields=snap), got, corners, win, steps, f"after {n_before} steps")


def _corners(n, win):
    # bulk (crossing a 56- and a 120-column strip seam and a chunk seam), face (periodic x edge), wrap corner
    return [(n // 2 - 20, n // 2 - 30), (n - win // 2, n // 3), (n - win // 2, n - win // 2)]


# ---- cfg2 4096^2 (20 steps full grid, both precisions; segments at steps 5000 and 9980) ------------------
@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg2_4096_full_grid_20_steps(prec):
    w = wl.cfg2(n=4096, prec=prec)
    g = make_gpu(w)
    g.step_rk4(20)
    got = g.read_field("psi_p")
    g.destroy()
    o = make_oracle(w)
    o.step_rk4(20)
    check_close(got, o.psi_p, TOL[prec], f"{w.name} psi_p full grid, 20 steps")


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg2_4096_windows(prec):
    w = wl.cfg2(n=4096, prec=prec)
    _check_windows(w, _corners(4096, 64), 64, 8)


@pytest.mark.parametrize("prec,n_before", [("c32", 5000), ("c32", 9980), ("c64", 9980)])
def test_cfg2_4096_segment(prec, n_before):
    _check_windows_from_checkpoint(wl.cfg2(n=4096, prec=prec), n_before, _corners(4096, 64), 64, 20)


# ---- cfg3 4096^2 (10-step segments from GPU checkpoints at steps 0, 10 000, 49 990) -------------------------------------
def test_cfg3_4096_windows():
    w = wl.cfg3(n=4096, prec="c32")
    _check_windows(w, _corners(4096, 64), 64, 10)


@pytest.mark.parametrize("n_before", [10000, 49990])
def test_cfg3_4096_segment(n_before):
    # the pumped reservoir has built up and the condensate has grown by then (n0 = 0, psi0 = noise at the start)
    _check_windows_from_checkpoint(wl.cfg3(n=4096, prec="c32"), n_before, _corners(4096, 64), 64, 10)


# ---- cfg4 16384^2 (256^2 windows at the centre, a face and the wrap corner, 16 steps) -------------------------------------
def test_cfg4_16384_windows():
    w = wl.cfg4(n=16384, prec="c32")       # 2 x 2 GiB of state, 16 GiB of workspace planes
    _check_windows(w, _corners(16384, 256), 256, 16)


# ---- cfg5 512 x 256^2 ------------------------------------------------------------------------------------------------------
def test_cfg5_full_ensemble():
    w = wl.cfg5(n=256, batch=512, prec="c32")
    g = make_gpu(w)
    # integer noise stream of every cell of every realisation, first, second and last step of the 20 000
    for step in (0, 1, 19999):
        assert np.array_equal(g.debug_noise_u32(step), orc.noise_u32(256, 256, 512, w.seed, step)), f"step {step}"
    n_steps = 3
    g.step_rk4(n_steps)
    o = make_oracle(w)
    o.step_rk4(n_steps)
    for name in w.fields:
        got = g.read_field(name)
        ref = getattr(o, name)
        for r in range(w.batch):
            check_close(got[r], ref[r], TOL["c32"], f"realisation {r} {name}")
    check_close(g.ensemble_mean_density("psi_p"), o.ensemble_mean_density("psi_p"), TOL["c32"], "ensemble mean")
    g.destroy()


def test_cfg5_realisations_0_255_511_for_500_steps():
    """fields of realisations 0, 255, 511 after 500 noisy steps of the full 512 x 256^2 ensemble."""
    w = wl.cfg5(n=256, batch=512, prec="c32")
    g = make_gpu(w)
    g.step_rk4(500)
    got = {name: g.read_field(name) for name in w.fields}
    g.destroy()
    for r in (0, 255, 511):
        # the realisation index keys the noise: a batch of one whose key word 1 is r (orc_problem.first_realisation)
        o = orc.Oracle(w.nx, w.ny, w.dx, w.dy, orc.make_params(**w.params), model=w.model, batch=1, prec32=True,
                       noise=True, seed=w.seed, P=w.P.astype(np.float64), first_realisation=r)
        for name, arr in w.fields.items():
            o.set_field(name, arr[r:r + 1])
        o.step_rk4(500)
        for name in w.fields:
            err = check_close(got[name][r], getattr(o, name)[0], TOL["c32"], f"realisation {r} {name} after 500 steps")
            _report(f"cfg5_512x256_r{r}_{name}_500", err)


def test_cfg5_ensemble_mean_of_16_realisations_for_200_steps():
    w = wl.cfg5(n=256, batch=16, prec="c32")        # realisations 0..15 of the ensemble (same seeds, same noise keys)
    g = make_gpu(w)
    o = make_oracle(w)
    g.step_rk4(200)
    o.step_rk4(200)
    for name in w.fields:
        _report(f"cfg5_16x256_{name}_200", check_close(g.read_field(name), getattr(o, name), TOL["c32"], f"{w.name} {name} after 200 steps"))
    _report("cfg5_16x256_mean_200", check_close(g.ensemble_mean_density("psi_p"), o.ensemble_mean_density("psi_p"), TOL["c32"],
                                                "ensemble mean, 200 steps"))
    g.destroy()


def test_cfg5_last_steps_of_the_run():
    w = wl.cfg5(n=256, batch=512, prec="c32")
    n_before, n_last = w.n_steps - 2, 2          # steps 19 998 and 19 999 of the 20 000
    g = make_gpu(w)
    g.step_rk4(n_before)
    snap = {name: g.read_field(name) for name in w.fields}
    g.step_rk4(n_last)
    assert g.get_step() == w.n_steps
    o = make_oracle(w)
    for name, arr in snap.items():
        assert np.all(np.isfinite(arr)), name
        o.set_field(name, arr)
    o.step = n_before                            # the step index keys the noise
    o.step_rk4(n_last)
    for name in w.fields:
        got, ref = g.read_field(name), getattr(o, name)
        for r in range(w.batch):
            check_close(got[r], ref[r], TOL["c32"], f"realisation {r} {name}, last steps")
    g.destroy()
