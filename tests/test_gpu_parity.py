"""GPU parity of variant STAGE (one fused kernel per RK stage): libphx (CUDA, through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): relative L2 <= 1e-12 (complex fp64), <= 2e-5 (complex fp32);
Philox words bit-exact.  Sizes span several tiles plus a ragged tail (block tile: 256 x rows cells)."""
import numpy as np
import pytest

from paper_2411_18341_b200 import workloads as wl
import functools

import helpers
from helpers import TOL, compare, make_oracle, rel_l2

pytestmark = pytest.mark.gpu
STAGE = 1
make_gpu = functools.partial(helpers.make_gpu, variant=STAGE)   # AUTO resolves to the fused step (test_gpu_step_variant.py)


def run_pair(w, n_steps, **kw):
    g = make_gpu(w, **kw)
    o = make_oracle(w, **{k: v for k, v in kw.items() if k in ("bc", "E", "extra_params")})
    g.step_rk4(n_steps)
    o.step_rk4(n_steps)
    errs = compare(g, o, w)
    g.destroy()
    return errs


def test_cfg1_full_run_fp64():
    w = wl.cfg1()
    errs = run_pair(w, w.n_steps)
    assert errs["psi_p"] <= 1e-12


@pytest.mark.parametrize("prec", ["c32", "c64"])
@pytest.mark.parametrize("nx,ny", [(600, 75), (514, 40), (201, 67), (64, 64)])
def test_cfg2_reduced(prec, nx, ny):
    # several 256-wide tiles plus ragged tails in x and y; odd nx exercises the unvectorised path
    w = wl.cfg2(n=nx, ny=ny, prec=prec)
    run_pair(w, 100)


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


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_coherent_drive(prec):
    w = wl.cfg2(n=140, ny=90, prec=prec)
    rng = np.random.default_rng(30)
    E = (0.05 * (rng.standard_normal((w.ny, w.nx)) + 1j * rng.standard_normal((w.ny, w.nx)))).astype(
        np.complex64 if prec == "c32" else np.complex128)
    run_pair(w, 100, E=E, extra_params=dict(omega=3.7))


def test_density_offset():
    w = wl.cfg2(n=128, ny=64, prec="c64")
    run_pair(w, 50, extra_params=dict(density_offset=0.02))


# ---- stochastic path ---------------------------------------------------------------------------------
def test_philox_words_bit_exact():
    import oracle as orc
    w = wl.cfg5(n=64, batch=5)
    g = make_gpu(w)
    for step in (0, 1, 19999, (3 << 32) + 17):
        got = g.debug_noise_u32(step)
        ref = orc.noise_u32(w.nx, w.ny, w.batch, w.seed, step)
        assert np.array_equal(got, ref)
    g.destroy()


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_cfg5_noisy_ensemble_reduced(prec):
    w = wl.cfg5(n=64, batch=6, prec=prec)
    g = make_gpu(w)
    o = make_oracle(w)
    g.step_rk4(60)
    o.step_rk4(60)
    compare(g, o, w)
    mean = g.ensemble_mean_density("psi_p")
    assert rel_l2(mean, o.ensemble_mean_density("psi_p")) <= TOL[prec]
    g.destroy()


def test_noise_one_step_from_zero_matches_normal_map():
    # psi = 0, n = 0: after one step psi is exactly sigma*(xi1 + i xi2); checks the float Box-Muller per cell
    w = wl.cfg5(n=64, batch=3, prec="c32")
    w.fields["psi_p"][...] = 0
    g = make_gpu(w)
    o = make_oracle(w)
    g.step_rk4(1)
    o.step_rk4(1)
    got = g.read_field("psi_p")
    assert np.max(np.abs(got - o.psi_p)) <= 4e-7 * np.max(np.abs(o.psi_p))
    g.destroy()


def test_spinor_noise():
    w = wl.cfg4(n=96, prec="c32", sigma_cells=10.0)
    w.noise, w.seed = True, 11
    run_pair(w, 30)


# ---- GPU-only invariants (no oracle) --------------------------------------------------------------------
@pytest.mark.parametrize("model", ["scalar", "reservoir", "spinor", "spinor_reservoir"])
def test_shift_equivariance_bit_exact(model):
    maker = {"scalar": lambda: wl.cfg2(n=300, ny=70, prec="c32"), "reservoir": lambda: wl.cfg3(n=200, prec="c32"),
             "spinor": lambda: wl.cfg4(n=200, prec="c32", sigma_cells=15.0), "spinor_reservoir": lambda: wl.example3(n=140)}[model]
    w = maker()
    g = make_gpu(w)
    g.step_rk4(10)
    base = {k: g.read_field(k) for k in w.fields}
    g.destroy()
    sh = (37, -4)   # (rows, cols); the column shift is even so that 128-bit alignment classes are preserved
    w2 = maker()
    for k in w2.fields:
        w2.fields[k] = np.ascontiguousarray(np.roll(w2.fields[k], sh, (1, 2)))
    if w2.V is not None:
        w2.V = np.ascontiguousarray(np.roll(w2.V, sh, (0, 1)))
    if w2.P is not None:
        w2.P = np.ascontiguousarray(np.roll(w2.P, sh, (0, 1)))
    g2 = make_gpu(w2)
    g2.step_rk4(10)
    for k in w.fields:
        assert np.array_equal(np.roll(base[k], sh, (1, 2)), g2.read_field(k)), k
    g2.destroy()


def test_step_splitting_is_bit_exact_with_noise():
    w = wl.cfg5(n=64, batch=3)
    g1, g2 = make_gpu(w), make_gpu(w)
    g1.step_rk4(23)
    for n in (1, 8, 9, 5):
        g2.step_rk4(n)
    assert g1.get_step() == g2.get_step() == 23
    for k in w.fields:
        assert np.array_equal(g1.read_field(k), g2.read_field(k))
    g1.destroy()
    g2.destroy()


def test_checkpoint_restart_is_bit_exact():
    w = wl.cfg5(n=64, batch=2)
    g1 = make_gpu(w)
    g1.step_rk4(7)
    snap = {k: g1.read_field(k) for k in w.fields}
    g1.step_rk4(5)
    g2 = make_gpu(w)
    for k, v in snap.items():
        g2.set_field(k, v)
    g2.set_step(7)
    g2.step_rk4(5)
    for k in w.fields:
        assert np.array_equal(g1.read_field(k), g2.read_field(k))
    g1.destroy()
    g2.destroy()


def test_tuning_rows_and_vec_do_not_change_results():
    w = wl.cfg3(n=192, prec="c32")
    outs = []
    for tuning in ({"rows": 16}, {"rows": 5}, {"rows": 64, "vec": 1}):
        g = make_gpu(w, tuning=tuning)
        g.step_rk4(20)
        outs.append({k: g.read_field(k) for k in w.fields})
        g.destroy()
    for k in w.fields:
        assert np.array_equal(outs[0][k], outs[1][k]) and np.array_equal(outs[0][k], outs[2][k])


def test_device_buffers_and_api_errors():
    import torch
    from paper_2411_18341_b200 import binding as phx
    w = wl.cfg2(n=128, ny=64, prec="c32")
    g = phx.Grid(w.nx, w.ny, w.dx, w.dy)
    g.select_variant(STAGE)
    with pytest.raises(phx.PhxError) as e:
        g.step_rk4(1)
    assert e.value.status == phx.PHX_ERR_BAD_STATE
    with pytest.raises(phx.PhxError) as e:
        g.set_field("n_p", np.zeros((1, w.ny, w.nx), np.float32))
    assert e.value.status == phx.PHX_ERR_UNSUPPORTED
    with pytest.raises(phx.PhxError) as e:         # a pump needs a reservoir (Eq. (17))
        g.set_potential_pump(None, np.ones((w.ny, w.nx), np.float32))
    assert e.value.status == phx.PHX_ERR_UNSUPPORTED
    assert g.set_params(phx.make_params(dt=1.0)) == phx.PHX_WARN_UNSTABLE
    assert g.set_params(phx.make_params(**w.params)) == phx.PHX_OK
    dev_psi = torch.from_numpy(w.fields["psi_p"]).cuda()
    dev_V = torch.from_numpy(w.V).cuda()
    g.set_potential_pump(dev_V, None)
    g.set_field("psi_p", dev_psi)
    g.step_rk4(10)
    out = torch.empty_like(dev_psi)
    g.read_field("psi_p", out)
    g2 = make_gpu(w)
    g2.step_rk4(10)
    assert np.array_equal(out.cpu().numpy(), g2.read_field("psi_p"))
    assert g.get_launch_count() == 40
    c = g.get_coeffs()
    assert np.array_equal(c, c.astype(np.float32).astype(np.float64)) and abs(c[0] - 25.0) < 1e-5
    g.destroy()
    g2.destroy()


def test_check_finite_reports_nan_and_inf_in_any_state_field():
    """phx_check_finite: finite fields -> True; one NaN / Inf anywhere in psi or n of any realisation ->
    False; an RK4 run far beyond its stability limit (PHX_WARN_UNSTABLE) ends non-finite and is caught."""
    w = wl.cfg5(n=64, batch=3, prec="c32")
    for variant in (1, 3):
        g = make_gpu(w, variant=variant)
        g.step_rk4(3)
        assert g.check_finite()
        n = g.read_field("n_p")
        n[2, 63, 63] = np.inf
        g.set_field("n_p", n)
        assert not g.check_finite()
        n[2, 63, 63] = 0.0
        g.set_field("n_p", n)
        psi = g.read_field("psi_p")
        psi[1, 17, 5] = complex(0.0, np.nan)
        g.set_field("psi_p", psi)
        assert not g.check_finite()
        g.destroy()
    w2 = wl.cfg2(n=64, ny=48, prec="c64")
    g = make_gpu(w2, extra_params=dict(dt=0.4))         # (hbar/2m)(8/dx^2) dt = 80 >> 2.78
    g.step_rk4(400)
    assert not g.check_finite()
    g.destroy()
