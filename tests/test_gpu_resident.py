"""GPU parity of variant RESIDENT (a grid of at most 64 x 64 cells stays on chip for all steps of one launch;
DESIGN.md section 5.3) against the CPU oracle, element by element, plus the invariants that need no oracle.
Bars as everywhere (BASELINE.json north_star): relative L2 <= 1e-12 (complex fp64), <= 2e-5 (complex fp32)."""
import dataclasses

import numpy as np
import pytest

from paper_2411_18341_b200 import binding as phx
from paper_2411_18341_b200 import workloads as wl
from helpers import TOL, compare, make_gpu, make_oracle, rel_l2

pytestmark = pytest.mark.gpu
STAGE, STEP, RESIDENT = 1, 3, 4


def run_pair(w, n_steps, **kw):
    g = make_gpu(w, variant=RESIDENT, **kw)
    assert g.get_variant() == RESIDENT
    o = make_oracle(w, **{k: v for k, v in kw.items() if k in ("bc", "extra_params")})
    g.step_rk4(n_steps)
    o.step_rk4(n_steps)
    errs = compare(g, o, w)
    assert g.get_launch_count() == 1               # all steps in one launch
    assert g.get_step() == n_steps
    g.destroy()
    return errs


def test_cfg1_full_run():
    w = wl.cfg1()                                  # 64 x 64, fp64, 1000 steps: BASELINE configs[0]
    g = make_gpu(w, variant=RESIDENT)
    assert g.get_variant() == RESIDENT
    o = make_oracle(w)
    g.step_rk4(w.n_steps)
    o.step_rk4(w.n_steps)
    errs = compare(g, o, w)
    assert errs["psi_p"] <= 1e-12
    g.destroy()


@pytest.mark.parametrize("prec", ["c32", "c64"])
@pytest.mark.parametrize("nx,ny", [(64, 64), (50, 41), (33, 7), (8, 5), (5, 4)])
def test_scalar(prec, nx, ny):
    run_pair(wl.cfg2(n=nx, ny=ny, prec=prec), 101)


@pytest.mark.parametrize("prec,n", [("c32", 64), ("c32", 37), ("c64", 45), ("c64", 20)])
def test_reservoir(prec, n):
    run_pair(wl.cfg3(n=n, prec=prec), 200)


@pytest.mark.parametrize("bc", [(1, 1), (1, 0), (0, 1)])
@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_zero_boundaries_and_anisotropic_grid(bc, prec):
    w = wl.cfg2(n=52, ny=31, prec=prec)
    run_pair(dataclasses.replace(w, dy=w.dx * 1.3), 60, bc=bc)


def test_density_offset():
    run_pair(wl.cfg2(n=48, ny=32, prec="c64"), 50, extra_params=dict(density_offset=0.02))


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_noisy_ensemble(prec):
    w = wl.cfg5(n=48 if prec == "c32" else 40, batch=33, prec=prec)
    g = make_gpu(w)
    assert g.get_variant() == RESIDENT             # AUTO: an ensemble (batch >= 32) of grids that fit
    o = make_oracle(w)
    g.step_rk4(40)
    o.step_rk4(40)
    compare(g, o, w)
    assert rel_l2(g.ensemble_mean_density("psi_p"), o.ensemble_mean_density("psi_p")) <= TOL[prec]
    g.destroy()


def test_step_splitting_checkpoint_and_variant_switches_are_consistent():
    w = wl.cfg5(n=40, batch=3)
    g1, g2 = make_gpu(w, variant=RESIDENT), make_gpu(w, variant=RESIDENT)
    g1.step_rk4(23)
    for n in (1, 8, 9, 5):
        g2.step_rk4(n)
    for k in w.fields:                             # the step counter keys the noise: k calls of one step == one call of k
        assert np.array_equal(g1.read_field(k), g2.read_field(k))
    # RESIDENT -> STEP (odd number of steps: ping-pong parity) -> RESIDENT -> STAGE, against the oracle
    g1.select_variant(STEP)
    g1.step_rk4(3)
    g1.select_variant(RESIDENT)
    g1.step_rk4(4)
    g1.select_variant(STAGE)
    g1.step_rk4(2)
    o = make_oracle(w)
    o.step_rk4(32)
    compare(g1, o, w)
    assert g1.get_step() == 32
    g1.destroy()
    g2.destroy()


def test_resident_agrees_with_step_to_rounding():
    w = wl.cfg3(n=44, prec="c64")
    a, b = make_gpu(w, variant=RESIDENT), make_gpu(w, variant=STEP)
    a.step_rk4(50)
    b.step_rk4(50)
    for k in w.fields:
        assert rel_l2(a.read_field(k), b.read_field(k)) <= 1e-13
    a.destroy()
    b.destroy()


def test_grids_that_do_not_fit_are_refused():
    for w, kw in ((wl.cfg2(n=256, ny=256, prec="c32"), {}), (wl.cfg4(n=32, prec="c32", sigma_cells=5.0), {}),
                  (wl.cfg2(n=128, ny=65, prec="c32"), {})):   # too many cells even for a cluster; spinor; too many cells for one CTA and an odd row count
        g = make_gpu(w, **kw)
        assert g.get_variant() == STEP
        with pytest.raises(phx.PhxError) as e:
            g.select_variant(RESIDENT)
        assert e.value.status == phx.PHX_ERR_UNSUPPORTED
        g.destroy()
    w = wl.cfg2(n=32, ny=32, prec="c32")
    g = make_gpu(w)
    assert g.get_variant() == RESIDENT             # AUTO: a single small grid runs on a cluster (the cluster form)
    g.set_drive(np.zeros((32, 32), np.complex64))  # a drive on a scalar grid: the cluster form carries it
    assert g.get_variant() == RESIDENT
    g.destroy()
    g = make_gpu(wl.cfg3(n=32, prec="c32"))
    assert g.get_variant() == RESIDENT
    g.set_drive(np.zeros((32, 32), np.complex64))  # a drive on a reservoir grid: the fused step takes over
    assert g.get_variant() == STEP
    g.destroy()
    g = make_gpu(wl.cfg2(n=33, ny=31, prec="c32"))
    assert g.get_variant() == STEP                 # an odd row count has no cluster form: the fused step spreads it over several SMs
    g.select_variant(RESIDENT)
    assert g.get_variant() == RESIDENT             # (one CTA, on request)
    g.destroy()


def _noisy(w):
    w.noise, w.seed = True, 13
    w.params = dict(w.params, noise_scale=1e-6)
    return w


# ---- cluster form: one realisation on a thread-block cluster of 2-16 CTAs ------------------------------
@pytest.mark.parametrize("maker,bc", [
    (lambda: wl.cfg1(n_steps=100), (0, 0)),                               # 64 x 64 fp64: 8 CTAs of 8 rows, one cell per thread
    (lambda: wl.cfg2(n=64, ny=64, prec="c32"), (0, 0)),
    (lambda: wl.cfg2(n=128, ny=128, prec="c32"), (0, 0)),                 # 16 rows per CTA, four cells per thread
    (lambda: wl.cfg2(n=128, ny=128, prec="c64"), (1, 1)),
    (lambda: wl.cfg2(n=96, ny=40, prec="c32"), (0, 1)),                   # 5 rows per CTA; zero boundary in y
    (lambda: wl.cfg2(n=50, ny=12, prec="c64"), (1, 0)),                   # 12 rows: a cluster of 4
    (lambda: wl.cfg2(n=33, ny=6, prec="c32"), (0, 0)),                    # 6 rows: a cluster of 2, the neighbour above is the neighbour below
    (lambda: wl.cfg3(n=64, prec="c32"), (0, 0)),
    (lambda: wl.cfg3(n=128, prec="c64"), (0, 0)),
    (lambda: wl.cfg5(n=64, batch=3, prec="c32"), (0, 0)),                 # noise: the cell index of the counter is the grid's
    (lambda: wl.cfg5(n=128, batch=2, prec="c32"), (0, 0)),
    (lambda: _noisy(wl.cfg2(n=64, ny=64, prec="c32")), (0, 0)),           # scalar + noise: the two-stages-per-barrier kernel
    (lambda: _noisy(wl.cfg2(n=40, ny=24, prec="c64")), (1, 1)),
    (lambda: wl.cfg2(n=33, ny=6, prec="c64"), (0, 0)),                    # an odd number of cells per slab in fp64
    (lambda: wl.cfg2(n=35, ny=10, prec="c64"), (0, 1)),
    (lambda: wl.cfg3(n=34, prec="c64"), (0, 0))])
def test_cluster_form(maker, bc):
    w = maker()
    g = make_gpu(w, variant=RESIDENT, bc=bc, tuning={"resident_cluster": 1})
    assert g.get_variant() == RESIDENT
    o = make_oracle(w, bc=bc)
    g.step_rk4(57)
    g.step_rk4(4)
    o.step_rk4(61)
    compare(g, o, w)
    assert g.get_launch_count() == 2 and g.get_step() == 61
    # (scalar grids run resident_pair_kernel: two stages per cluster barrier, one redundant row of arithmetic on either side)
    # against the one-CTA form where the grid fits it: the same cell arithmetic (phx_deriv.cuh), hence the same bits -- except
    # with noise, where the compiler contracts the reservoir / variance expressions differently for 1 and 8 cells per thread
    # (rounding-level: bounded at a tenth of the field tolerance)
    if w.nx * w.ny <= 4096 and not (w.prec == "c64" and w.model == "reservoir" and w.nx * w.ny > 2048):
        ref = make_gpu(w, variant=RESIDENT, bc=bc, tuning={"resident_cluster": 0})
        ref.step_rk4(61)
        for name in w.fields:
            if w.noise:
                assert rel_l2(g.read_field(name), ref.read_field(name)) <= 0.1 * TOL[w.prec], name
            else:
                assert np.array_equal(g.read_field(name), ref.read_field(name)), name
        ref.destroy()
    g.destroy()


def test_cluster_form_opens_resident_to_128_wide_grids():
    g = make_gpu(wl.cfg2(n=128, ny=128, prec="c32"))      # AUTO: does not fit one CTA; a cluster of 16 steps it faster than STEP
    assert g.get_variant() == RESIDENT
    g.destroy()
    g = make_gpu(wl.cfg2(n=192, ny=96, prec="c32"))       # AUTO beyond 128^2 cells: the fused step
    assert g.get_variant() == STEP
    g.select_variant(RESIDENT)
    assert g.get_variant() == RESIDENT                     # (the cluster form, on request)
    g.destroy()
    g = make_gpu(wl.cfg2(n=128, ny=128, prec="c32"), tuning={"resident_cluster": 0})
    with pytest.raises(phx.PhxError):
        g.select_variant(RESIDENT)                         # without the cluster form the request is refused
    g.destroy()



@pytest.mark.parametrize("prec,nx,ny,bc,noise", [("c64", 64, 64, (0, 0), False), ("c32", 128, 128, (0, 0), False), ("c32", 50, 24, (1, 0), False),
                                                  ("c64", 33, 6, (0, 1), False), ("c32", 64, 32, (0, 0), True)])
def test_cluster_form_with_coherent_drive(prec, nx, ny, bc, noise):
    """E(r) exp(-i omega t) at the stage times (reading Q17) in the cluster form of the scalar
    model (resident_pair_kernel): against the oracle, and against the fused step to a tenth of the tolerance; AUTO keeps a driven single small scalar grid in RESIDENT."""
    w = wl.cfg2(n=nx, ny=ny, prec=prec)
    if noise:
        w = _noisy(w)
    rng = np.random.default_rng(31)
    E = (0.05 * (rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx)))).astype(np.complex64 if prec == "c32" else np.complex128)
    xp = dict(omega=3.7)
    g = make_gpu(w, bc=bc, E=E, extra_params=xp)
    assert g.get_variant() == RESIDENT
    o = make_oracle(w, bc=bc, E=E, extra_params=xp)
    g.step_rk4(40)
    g.step_rk4(21)              # (the phase follows the step counter across calls)
    o.step_rk4(61)
    compare(g, o, w)
    ref = make_gpu(w, bc=bc, E=E, extra_params=xp, variant=STEP)
    ref.step_rk4(61)
    # (the fused step evaluates the isotropic, hbar = 1 form of the same derivative: rounding-level differences)
    assert rel_l2(g.read_field("psi_p"), ref.read_field("psi_p")) <= 0.1 * TOL[prec]
    g.destroy()
    ref.destroy()
