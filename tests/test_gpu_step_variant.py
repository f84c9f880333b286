"""GPU parity of variant STEP (one kernel per RK4 step, four stages temporally blocked in registers; DESIGN.md
section 5.2) against the CPU oracle, element by element, plus the invariants that need no oracle.
Bars as in test_gpu_parity.py (BASELINE.json north_star): relative L2 <= 1e-12 (complex fp64), <= 2e-5 (complex fp32).
Sizes span several warp strips (56 / 24 output columns per strip) and row chunks with ragged tails in x and y."""
import dataclasses

import numpy as np
import pytest

from paper_2411_18341_b200 import workloads as wl
from helpers import TOL, compare, make_gpu, make_oracle, rel_l2

pytestmark = pytest.mark.gpu
STEP, STAGE = 3, 1


def run_pair(w, n_steps, tuning=None, **kw):
    g = make_gpu(w, variant=STEP, tuning=tuning, **kw)
    assert g.get_variant() == STEP
    o = make_oracle(w, **{k: v for k, v in kw.items() if k in ("bc", "E", "extra_params")})
    g.step_rk4(n_steps)
    o.step_rk4(n_steps)
    errs = compare(g, o, w)
    assert g.get_launch_count() in (n_steps, 2 * n_steps)   # one kernel per RK4 step (two when a ragged last strip has its side launch)
    g.destroy()
    return errs


def test_cfg1_full_run_fp64():
    w = wl.cfg1()
    errs = run_pair(w, w.n_steps)
    assert errs["psi_p"] <= 1e-12


@pytest.mark.parametrize("prec", ["c32", "c64"])
@pytest.mark.parametrize("nx,ny", [(600, 75), (514, 40), (201, 67), (64, 64), (56, 9), (8, 5)])
def test_cfg2_reduced(prec, nx, ny):
    # odd nx runs one cell per lane; nx < strip width wraps a strip onto itself
    w = wl.cfg2(n=nx, ny=ny, prec=prec)
    run_pair(w, 101)                               # odd count: the state ends in the alternate buffer


@pytest.mark.parametrize("tuning", [{"step_ly": 8}, {"step_ly": 13, "step_vec": 1}, {"step_ly": 1000},
                                    {"step_ly": 13, "step_vec": 4}, {"step_vec": 4}])
def test_cfg2_chunking(tuning):
    w = wl.cfg2(n=300, ny=70, prec="c32")
    run_pair(w, 60, tuning=tuning)


@pytest.mark.parametrize("prec", ["c32", "c64"])
@pytest.mark.parametrize("model", ["scalar", "reservoir", "spinor_reservoir"])
def test_anisotropic_grid(prec, model):
    # dx != dy: the general form of the Laplacian (cx != cy); every other STEP case here has dx == dy
    w = {"scalar": lambda: wl.cfg2(n=300, ny=70, prec=prec), "reservoir": lambda: wl.cfg3(n=96, prec=prec),
         "spinor_reservoir": lambda: wl.example3(n=90, prec=prec)}[model]()
    w = dataclasses.replace(w, dy=w.dx * 1.25)
    run_pair(w, 60)
    if model == "scalar" and prec == "c32":
        run_pair(w, 60, tuning={"step_vec": 4})


@pytest.mark.parametrize("tuning", [{"step_vec": 2}, {"step_vec": 2, "step_ly": 11}])
def test_cfg2_fp64_two_cells_per_lane(tuning):
    w = wl.cfg2(n=300, ny=70, prec="c64")
    run_pair(w, 60, tuning=tuning)
    run_pair(dataclasses.replace(w, dy=w.dx * 0.8), 40, tuning=tuning)      # general (dx != dy) form
    run_pair(wl.cfg2(n=132, ny=70, prec="c64"), 40, bc=(1, 1), tuning=tuning)   # zero boundaries


def test_wide_scalar_grid_takes_four_cells_per_lane():
    w = wl.cfg2(n=2048, ny=48, prec="c32")
    g = make_gpu(w, variant=STEP)
    o = make_oracle(w)
    g.step_rk4(30)
    o.step_rk4(30)
    compare(g, o, w)
    g.destroy()


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg2_1024_horizon(prec):
    w = wl.cfg2(n=1024, prec=prec)
    run_pair(w, 40)


@pytest.mark.parametrize("prec", ["c32", "c64"])
@pytest.mark.parametrize("n", [96, 300])
def test_cfg3_reservoir_reduced(prec, n):
    w = wl.cfg3(n=n, prec=prec)
    run_pair(w, 200)


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg4_spinor_reduced(prec):
    w = wl.cfg4(n=320, prec=prec, sigma_cells=20.0)
    run_pair(w, 100)


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_spinor_reservoir_example3(prec):
    w = wl.example3(n=150, prec=prec)
    run_pair(w, 100)


@pytest.mark.parametrize("bc", [(1, 1), (1, 0), (0, 1)])
@pytest.mark.parametrize("model", ["scalar", "spinor_reservoir"])
def test_zero_boundaries(bc, model):
    w = wl.cfg2(n=130, ny=70, prec="c64") if model == "scalar" else wl.example3(n=90, prec="c64")
    run_pair(w, 50, bc=bc)


@pytest.mark.parametrize("vec", [2, 4])
def test_zero_boundaries_fp32_cells_per_lane(vec):
    w = wl.cfg2(n=132, ny=70, prec="c32")
    run_pair(w, 50, bc=(1, 1), tuning={"step_ly": 16, "step_vec": vec})


def test_density_offset():
    w = wl.cfg2(n=128, ny=64, prec="c64")
    run_pair(w, 50, extra_params=dict(density_offset=0.02))


def _drive_field(w, seed=30):
    rng = np.random.default_rng(seed)
    return (0.05 * (rng.standard_normal((w.ny, w.nx)) + 1j * rng.standard_normal((w.ny, w.nx)))).astype(
        np.complex64 if w.prec == "c32" else np.complex128)


@pytest.mark.parametrize("prec", ["c32", "c64"])
@pytest.mark.parametrize("model", ["scalar", "reservoir", "spinor", "spinor_reservoir"])
def test_coherent_drive(prec, model):
    # E(r) exp(-i omega t) at the stage times t, t + dt/2, t + dt (reading Q17)
    w = {"scalar": lambda: wl.cfg2(n=140, ny=90, prec=prec), "reservoir": lambda: wl.cfg3(n=96, prec=prec),
         "spinor": lambda: wl.cfg4(n=96, prec=prec, sigma_cells=10.0), "spinor_reservoir": lambda: wl.example3(n=90, prec=prec)}[model]()
    run_pair(w, 101, E=_drive_field(w), extra_params=dict(omega=3.7))


@pytest.mark.parametrize("tuning,bc", [({"step_vec": 4}, (0, 0)), ({"step_vec": 2, "step_ly": 9}, (1, 1)), ({"step_vec": 1}, (0, 1))])
def test_coherent_drive_cells_per_lane_and_boundaries(tuning, bc):
    w = wl.cfg2(n=132, ny=70, prec="c32")
    w = dataclasses.replace(w, dy=w.dx * 1.1)
    run_pair(w, 60, E=_drive_field(w), extra_params=dict(omega=-2.1), tuning=tuning, bc=bc)


def test_drive_set_mid_run_and_drive_with_noise():
    w = wl.cfg2(n=64, ny=32, prec="c32")
    E = _drive_field(w)
    xp = dict(omega=1.3)
    g = make_gpu(w, variant=STEP, extra_params=xp)
    g.step_rk4(3)                                  # odd: state in the alternate buffer
    g.set_drive(E)                                 # the fused step carries on, now with the drive
    assert g.get_variant() == STEP
    g.step_rk4(2)
    o = make_oracle(w, extra_params=xp)
    o.step_rk4(3)
    o2 = make_oracle(w, E=E, extra_params=xp)
    o2.set_field("psi_p", o.psi_p)
    o2.step = 3
    o2.step_rk4(2)
    assert rel_l2(g.read_field("psi_p"), o2.psi_p) <= TOL["c32"]
    g.destroy()
    # Eq. (16) carries E and dW together: a driven grid with noise runs the fused step as well
    for wn in (wl.cfg5(n=64, batch=2), dataclasses.replace(wl.cfg4(n=96, prec="c32", sigma_cells=10.0), noise=True, seed=11)):
        En = _drive_field(wn)
        gn = make_gpu(wn, E=En, extra_params=xp)
        assert gn.get_variant() == STEP
        on = make_oracle(wn, E=En, extra_params=xp)
        gn.step_rk4(25)
        on.step_rk4(25)
        compare(gn, on, wn)
        gn.destroy()


# ---- stochastic path -------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg5_noisy_ensemble_reduced(prec):
    w = wl.cfg5(n=64, batch=6, prec=prec)
    g = make_gpu(w, variant=STEP)
    o = make_oracle(w)
    g.step_rk4(61)
    o.step_rk4(61)
    compare(g, o, w)
    mean = g.ensemble_mean_density("psi_p")
    assert rel_l2(mean, o.ensemble_mean_density("psi_p")) <= TOL[prec]
    g.destroy()


def test_noise_one_step_from_zero_matches_normal_map():
    # psi = 0, n = 0: after one step psi is exactly sigma (xi1 + i xi2): the float Box-Muller map, cell by cell.
    # The fused kernels evaluate it on the special-function unit (phx_philox.cuh, noise_increment_sfu): lg2.approx has a
    # relative error of 2^-22, sin.approx / cos.approx an absolute error of 2^-20.9 = 5.1e-7 on [-pi, pi] (PTX ISA), and
    # the angle 2 pi (u2 - 1/2) is rounded once (1.9e-7): an element is within 1e-6 of its own radius of the
    # double-precision map, hence within 2e-6 of the largest one.  (The per-stage kernels keep logf / sincospif: 4e-7 there.)
    w = wl.cfg5(n=64, batch=3, prec="c32")
    w.fields["psi_p"][...] = 0
    g = make_gpu(w, variant=STEP)
    o = make_oracle(w)
    g.step_rk4(1)
    o.step_rk4(1)
    got = g.read_field("psi_p")
    assert np.max(np.abs(got - o.psi_p)) <= 2e-6 * np.max(np.abs(o.psi_p))
    assert rel_l2(got, o.psi_p) <= 1e-6
    g.destroy()


def test_spinor_noise():
    w = wl.cfg4(n=96, prec="c32", sigma_cells=10.0)
    w.noise, w.seed = True, 11
    run_pair(w, 30)


# ---- exchanging strips (the warps of a CTA tile the whole row), side launch, bulk-copy fetch ---------------
def _fields(g, w):
    return {name: g.read_field(name) for name in w.fields}


@pytest.mark.parametrize("prec,nx,vec", [("c32", 64, 2), ("c32", 128, 2), ("c32", 256, 2), ("c32", 512, 2), ("c32", 128, 4),
                                         ("c32", 1024, 4), ("c64", 32, 1), ("c64", 96, 1), ("c64", 256, 1), ("c64", 128, 2)])
def test_exchanging_strips_scalar(prec, nx, vec):
    # rows of 1, 2, 3, 4 and 8 strips; ragged chunks (ny = 45); against the oracle, and bit for bit against the independent
    # strips (the same cell arithmetic: only where a neighbour's value comes from differs)
    w = wl.cfg2(n=nx, ny=45, prec=prec)
    g = make_gpu(w, variant=STEP, tuning={"step_xch": 1, "step_vec": vec, "step_ly": 11})
    o = make_oracle(w)
    g.step_rk4(41)
    o.step_rk4(41)
    compare(g, o, w)
    ref = make_gpu(w, variant=STEP, tuning={"step_xch": 0, "step_vec": vec})
    ref.step_rk4(41)
    assert np.array_equal(g.read_field("psi_p"), ref.read_field("psi_p"))
    g.destroy()
    ref.destroy()


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_exchanging_strips_noisy_reservoir_ensemble(prec):
    # cfg5's shape in small: 4 strips of 64 columns (fp64: 8 of 32), several realisations, noise, odd step count
    w = wl.cfg5(n=256, batch=3, prec=prec)
    g = make_gpu(w, variant=STEP, tuning={"step_xch": 1, "step_ly": 37})
    o = make_oracle(w)
    g.step_rk4(25)
    o.step_rk4(25)
    compare(g, o, w)
    ref = make_gpu(w, variant=STEP, tuning={"step_xch": 0})
    ref.step_rk4(25)
    for name in w.fields:
        assert np.array_equal(g.read_field(name), ref.read_field(name)), name
    g.destroy()
    ref.destroy()


def test_exchanging_strips_are_the_default_for_ensembles_of_narrow_grids():
    # AUTO: a million cells or more in rows of at most four strips; same bits either way
    w = wl.cfg5(n=128, batch=64, prec="c32")
    g = make_gpu(w, variant=STEP)
    ref = make_gpu(w, variant=STEP, tuning={"step_xch": 0})
    g.step_rk4(7)
    ref.step_rk4(7)
    for name in w.fields:
        assert np.array_equal(g.read_field(name), ref.read_field(name)), name
    g.destroy()
    ref.destroy()


@pytest.mark.parametrize("maker", [lambda: wl.cfg1(n_steps=60), lambda: wl.cfg2(n=300, ny=70, prec="c32"), lambda: wl.cfg3(n=160, prec="c32"),
                                   lambda: wl.cfg4(n=120, prec="c32", sigma_cells=10.0), lambda: wl.cfg5(n=64, batch=5, prec="c32"),
                                   lambda: wl.cfg2(n=1024, ny=256, prec="c32")])
def test_programmatic_dependent_launches_give_the_same_bits(maker):
    # step_pdl: the later steps of a captured graph are programmatic dependents of the step before (griddepcontrol.wait at the
    # top of the kernel orders everything); forced on and off, odd and even step counts, noise counter included
    w = maker()
    on = make_gpu(w, variant=STEP, tuning={"step_pdl": 1})
    off = make_gpu(w, variant=STEP, tuning={"step_pdl": 0})
    for n in (19, 8, 1):
        on.step_rk4(n)
        off.step_rk4(n)
    for name in w.fields:
        assert np.array_equal(on.read_field(name), off.read_field(name)), name
    assert on.get_step() == off.get_step() == 28
    on.destroy()
    off.destroy()


@pytest.mark.parametrize("nx,bc,noise", [(2048, (0, 0), False), (2416, (0, 0), True), (4096, (0, 0), False), (2188, (1, 1), False),
                                         (2428, (0, 1), False)])
def test_side_launch_for_a_ragged_last_strip(nx, bc, noise):
    # 4 cells per lane: strips of 120 output columns; nx = k * 120 + (8, 16, 16, 28, 28): with step_side = 1 the remaining columns
    # are stepped by a side launch with one cell per lane on a second branch of the graph (measured
    # slower, hence opt-in).  Against the oracle, and bit for bit against the single launch; two kernels per step.
    w = wl.cfg2(n=nx, ny=37, prec="c32")
    if noise:
        w.noise, w.seed = True, 5
        w.params = dict(w.params, noise_scale=1e-6)
    g = make_gpu(w, variant=STEP, bc=bc, tuning={"step_vec": 4, "step_side": 1})
    ref = make_gpu(w, variant=STEP, bc=bc, tuning={"step_vec": 4})
    o = make_oracle(w, bc=bc)
    g.step_rk4(17)
    ref.step_rk4(17)
    o.step_rk4(17)
    compare(g, o, w)
    assert np.array_equal(g.read_field("psi_p"), ref.read_field("psi_p"))
    assert g.get_launch_count() == 34 and ref.get_launch_count() == 17
    g.destroy()
    ref.destroy()


@pytest.mark.parametrize("maker", [lambda: wl.cfg2(n=2048, ny=40, prec="c32"), lambda: wl.cfg2(n=300, ny=70, prec="c32"),
                                   lambda: wl.cfg2(n=200, ny=64, prec="c64"), lambda: wl.cfg3(n=160, prec="c32"),
                                   lambda: wl.cfg4(n=120, prec="c32", sigma_cells=10.0), lambda: wl.cfg5(n=64, batch=5, prec="c32")])
def test_bulk_copy_fetch_path(maker):
    # step_bulk = 1: rows fetched by TMA bulk copies into a shared-memory ring (profiles/r02_tma_vs_register_fetch.md);
    # the same cell arithmetic as the register loads: the same bits; strips that wrap around the periodic edge included
    w = maker()
    g = make_gpu(w, variant=STEP, tuning={"step_bulk": 1, "step_xch": 0})
    ref = make_gpu(w, variant=STEP, tuning={"step_xch": 0})
    o = make_oracle(w)
    g.step_rk4(23)
    ref.step_rk4(23)
    o.step_rk4(23)
    compare(g, o, w)
    for name in w.fields:
        assert np.array_equal(g.read_field(name), ref.read_field(name)), name
    g.destroy()
    ref.destroy()


# ---- invariants (no oracle) --------------------------------------------------------------------------------
@pytest.mark.parametrize("model", ["scalar", "reservoir", "spinor", "spinor_reservoir"])
def test_shift_equivariance_bit_exact(model):
    maker = {"scalar": lambda: wl.cfg2(n=300, ny=70, prec="c32"), "reservoir": lambda: wl.cfg3(n=200, prec="c32"),
             "spinor": lambda: wl.cfg4(n=200, prec="c32", sigma_cells=15.0), "spinor_reservoir": lambda: wl.example3(n=140)}[model]
    w = maker()
    g = make_gpu(w, variant=STEP)
    g.step_rk4(10)
    base = {k: g.read_field(k) for k in w.fields}
    g.destroy()
    sh = (37, -5)   # every cell is computed by the same instruction sequence whatever its lane, strip or chunk
    w2 = maker()
    for k in w2.fields:
        w2.fields[k] = np.ascontiguousarray(np.roll(w2.fields[k], sh, (1, 2)))
    if w2.V is not None:
        w2.V = np.ascontiguousarray(np.roll(w2.V, sh, (0, 1)))
    if w2.P is not None:
        w2.P = np.ascontiguousarray(np.roll(w2.P, sh, (0, 1)))
    g2 = make_gpu(w2, variant=STEP, tuning={"step_ly": 19})
    g2.step_rk4(10)
    for k in w.fields:
        assert np.array_equal(np.roll(base[k], sh, (1, 2)), g2.read_field(k)), k
    g2.destroy()
    if model == "scalar":   # four cells per lane: the same arithmetic per cell, so the same bits
        g4 = make_gpu(w2, variant=STEP, tuning={"step_vec": 4})
        g4.step_rk4(10)
        for k in w.fields:
            assert np.array_equal(np.roll(base[k], sh, (1, 2)), g4.read_field(k)), k
        g4.destroy()


def test_step_splitting_and_checkpoint_are_bit_exact_with_noise():
    w = wl.cfg5(n=64, batch=3)
    g1, g2 = make_gpu(w, variant=STEP), make_gpu(w, variant=STEP)
    g1.step_rk4(23)
    for n in (1, 8, 9, 5):
        g2.step_rk4(n)
    assert g1.get_step() == g2.get_step() == 23
    for k in w.fields:
        assert np.array_equal(g1.read_field(k), g2.read_field(k))
    # checkpoint at an odd step, restart in a fresh handle
    snap = {k: g1.read_field(k) for k in w.fields}
    g1.step_rk4(6)
    g3 = make_gpu(w, variant=STEP)
    for k, v in snap.items():
        g3.set_field(k, v)
    g3.set_step(23)
    g3.step_rk4(6)
    for k in w.fields:
        assert np.array_equal(g1.read_field(k), g3.read_field(k))
    for g in (g1, g2, g3):
        g.destroy()


def test_switching_variants_mid_run_keeps_state_and_noise_stream():
    w = wl.cfg5(n=64, batch=2)
    g = make_gpu(w, variant=STEP)
    g.step_rk4(5)
    g.select_variant(STAGE)
    g.step_rk4(4)
    g.select_variant(STEP)
    g.step_rk4(3)
    o = make_oracle(w)
    o.step_rk4(12)
    compare(g, o, w)
    assert g.get_step() == 12
    g.destroy()


def test_step_and_stage_agree_to_rounding():
    w = wl.cfg3(n=192, prec="c64")
    a, b = make_gpu(w, variant=STEP), make_gpu(w, variant=STAGE)
    a.step_rk4(50)
    b.step_rk4(50)
    for k in w.fields:
        assert rel_l2(a.read_field(k), b.read_field(k)) <= 1e-13
    a.destroy()
    b.destroy()


def test_async_host_copies_give_the_same_bits():
    # "async_host_copies": set_field / read_field enqueue the copy and return; phx_sync fences (bench.py's end-to-end leg)
    import torch
    w = wl.cfg2(n=300, ny=70, prec="c32")
    g = make_gpu(w, variant=STEP)
    g.step_rk4(3)
    ref = g.read_field("psi_p")
    g.destroy()
    pin_in = torch.from_numpy(np.ascontiguousarray(w.fields["psi_p"])).pin_memory()
    handles = [make_gpu(w, variant=STEP) for _ in range(2)]
    outs = [torch.empty_like(pin_in).pin_memory() for _ in handles]
    for h in handles:
        h.set_tuning("async_host_copies", 1)
    for rep in range(3):
        for h, out in zip(handles, outs):
            h.sync()
            h.set_field("psi_p", pin_in)
            h.set_step(0)
            h.step_rk4(3)
            h.read_field("psi_p", out)
    for h, out in zip(handles, outs):
        h.sync()
        assert np.array_equal(out.numpy().reshape(ref.shape), ref)
        h.destroy()
