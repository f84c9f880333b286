"""GPU parity of the adaptive Dormand-Prince 5(4) integrator (phx_step_adaptive, DESIGN.md
reading Q20) against the oracle's orc_step_dp54 on the same seeded inputs.

What is compared: the accept / reject flags and the quantised step factors q of EVERY attempt as integers, bit for bit (the
whole loop runs on the device: seven stage kernels, the max-norm reduction, the controller and the loop condition inside a
CUDA-graph WHILE node); the step sizes and error norms; and the fields at t_end within the north_star bars (relative L2
<= 1e-12 complex fp64, <= 2e-5 complex fp32, plus the element-wise guard).  Floating point decides the integers: each test
first checks, on the oracle's own log, that no decision sits within the kernel's rounding of its boundary."""
import dataclasses

import numpy as np
import pytest

from paper_2411_18341_b200 import binding as phx
from paper_2411_18341_b200 import workloads as wl
from helpers import TOL, check_close, make_oracle

pytestmark = pytest.mark.gpu
TOLS = {"c32": (1e-6, 1e-4), "c64": (1e-8, 1e-6)}      # (atol, rtol) of the error norm


def make_gpu(w, bc=(0, 0), E=None, extra_params=None):
    prm = dict(w.params)
    if extra_params:
        prm.update(extra_params)
    g = phx.Grid(w.nx, w.ny, w.dx, w.dy, model=w.model, prec=w.prec, batch=w.batch, noise=w.noise, bc=bc, integrator="dp54")
    g.set_params(phx.make_params(seed=w.seed, **prm))
    if w.V is not None or w.P is not None:
        g.set_potential_pump(w.V, w.P)
    if E is not None:
        g.set_drive(E)
    for name, arr in w.fields.items():
        g.set_field(name, arr)
    return g


def decision_margin(log):
    """Smallest relative distance of an error norm from a decision boundary (err = 1; 16 * 0.9 err^-1/5 an integer)."""
    err = log["err"]
    f = 16 * 0.9 * err ** -0.2
    inside = (f > 4.0) & (f < 64.0)                      # outside, the clamp decides and the margin is wide
    frac = np.minimum(f % 1.0, 1.0 - f % 1.0) / f
    return float(min(np.min(np.abs(err - 1.0)), np.min(np.where(inside, frac, 1.0)) * 5.0))


def run_pair(w, t_end, atol, rtol, h_init, h_max=1e30, check_sequence=True, **kw):
    g = make_gpu(w, **kw)
    o = make_oracle(w, **kw)
    g.step_adaptive(t_end, atol, rtol, h_init, h_max=h_max)
    lo = o.step_dp54(t_end, atol, rtol, h_init, h_max=h_max)
    st = g.get_adaptive_state()
    # how far the kernel's error norm may be from the oracle's: E = h sum e_j K_j cancels to 1e-4 of |h K| at these
    # tolerances, so complex fp32 carries it to a few 1e-4 relative (measured up to 3e-4), complex fp64 to 1e-12
    eps = 1e-3 if w.prec == "c32" else 1e-11
    if check_sequence:
        assert decision_margin(lo) > eps, "test case sits on a decision boundary: choose other parameters"
        assert st["attempts"] == lo["attempts"]
        assert np.array_equal(st["accept"], lo["accept"]), (st["accept"], lo["accept"])
        assert np.array_equal(st["q"], lo["q"]), (st["q"], lo["q"])
        assert np.array_equal(st["h"], lo["h"])              # same q sequence => bitwise the same step sizes
        big = lo["err"] > 0.02           # (an error norm far below 1 is rounding noise of the kernel's precision; q = 64 there)
        assert np.allclose(st["err"][big], lo["err"][big], rtol=eps)
        assert st["n_accept"] == o.ad.n_accept and st["n_reject"] == o.ad.n_reject
        assert st["h_next"] == o.ad.h_next
    assert st["t"] == t_end == o.ad.t
    for name in w.fields:
        check_close(g.read_field(name), getattr(o, name), TOL[w.prec], f"{w.name} {name} at t = {t_end}")
    g.destroy()
    return st, lo


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_scalar_cfg2_like(prec):
    w = wl.cfg2(n=200, ny=72, prec=prec)
    atol, rtol = TOLS[prec]
    st, lo = run_pair(w, 0.5, atol, rtol, 0.02, h_max=0.012)     # h_init > h_max: clamped; starts with rejections or growth
    assert st["attempts"] >= 40


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_reservoir_cfg3_like(prec):
    w = wl.cfg3(n=96, prec=prec)
    atol, rtol = TOLS[prec]
    # the first proposal is above the stability limit (omega_max h = 3.9): rejections.  The stiff grid takes 3000 attempts
    # per time unit; complex fp32 is run over a stretch whose decisions all keep the margin asked for in run_pair
    st, lo = run_pair(w, 0.03 if prec == "c32" else 0.2, atol, rtol, 2e-3)
    assert (lo["accept"] == 0).sum() >= 1 and st["attempts"] >= 80


@pytest.mark.parametrize("prec", ["c32", "c64"])
def test_spinor_and_spinor_reservoir(prec):
    atol, rtol = TOLS[prec]
    run_pair(wl.cfg4(n=96, prec=prec, sigma_cells=10.0), 0.3, atol, rtol, 0.01)
    run_pair(wl.example3(n=90, prec=prec), 0.25, atol, rtol, 0.002)


@pytest.mark.parametrize("bc", [(1, 1), (0, 1)])
def test_zero_boundaries_and_drive(bc):
    w = wl.cfg2(n=130, ny=70, prec="c64")
    w = dataclasses.replace(w, dy=w.dx * 1.2)
    rng = np.random.default_rng(31)
    E = (0.05 * (rng.standard_normal((w.ny, w.nx)) + 1j * rng.standard_normal((w.ny, w.nx)))).astype(np.complex128)
    run_pair(w, 0.4, 1e-9, 1e-7, 0.01, bc=bc, E=E, extra_params=dict(omega=3.7))


def test_batch_shares_one_step_size():
    w = wl.cfg5(n=64, batch=5, prec="c32", noise=False)
    run_pair(w, 0.3, *TOLS["c32"], 0.01)


def test_interrupted_and_resumed_run_and_mixing_with_rk4_steps():
    w = wl.cfg3(n=80, prec="c64")
    args = dict(atol=1e-9, rtol=1e-7, h_init=2e-3)
    a, b = make_gpu(w), make_gpu(w)
    a.step_adaptive(0.1, **args)
    b.step_adaptive(0.1, max_attempts=7, **args)
    sb = b.get_adaptive_state()
    assert sb["attempts"] == 7 and sb["t"] < 0.1
    b.step_adaptive(0.1, **args)
    sa, sb = a.get_adaptive_state(), b.get_adaptive_state()
    assert sa["t"] == sb["t"] == 0.1 and sa["h_next"] == sb["h_next"] and sa["n_accept"] == sb["n_accept"]
    for k in w.fields:
        assert np.array_equal(a.read_field(k), b.read_field(k))
    # fixed-step RK4 steps (an odd number: the fused step leaves the state in its alternate buffer) and adaptive stepping on
    # the same handle: the adaptive integrator picks the state up where phx_step_rk4 left it
    o = make_oracle(w)
    o.step_dp54(0.1, **args)
    a.step_rk4(3)
    o.step_rk4(3)
    a.step_adaptive(0.15, **args)
    o.step_dp54(0.15, **args)
    for k in w.fields:
        check_close(a.read_field(k), getattr(o, k), TOL["c64"], f"{k} after RK4 + adaptive")
    a.destroy()
    b.destroy()


def test_set_time_and_api_errors():
    w = wl.cfg2(n=64, ny=48, prec="c64")
    rng = np.random.default_rng(32)
    E = (0.05 * (rng.standard_normal((w.ny, w.nx)) + 1j * rng.standard_normal((w.ny, w.nx)))).astype(np.complex128)
    g = make_gpu(w, E=E, extra_params=dict(omega=2.0))
    g.set_time(1.7, 0.004)                                       # the drive phase follows the integrator's clock
    g.step_adaptive(1.9, 1e-9, 1e-7, 0.01)
    o = make_oracle(w, E=E, extra_params=dict(omega=2.0))
    o.ad.t, o.ad.h_next = 1.7, 0.004
    o.step_dp54(1.9, 1e-9, 1e-7, 0.01)
    check_close(g.read_field("psi_p"), o.psi_p, TOL["c64"], "after set_time")
    with pytest.raises(phx.PhxError) as e:
        g.step_adaptive(2.0, 0.0, 0.0, 0.01)
    assert e.value.status == phx.PHX_ERR_INVALID_ARG
    g.destroy()
    plain = phx.Grid(w.nx, w.ny, w.dx, w.dy, prec="c64")        # created without PHX_INT_DP54
    plain.set_params(phx.make_params(**w.params))
    with pytest.raises(phx.PhxError) as e:
        plain.step_adaptive(0.1, 1e-8, 1e-6, 0.01)
    assert e.value.status == phx.PHX_ERR_UNSUPPORTED
    plain.destroy()
    wn = wl.cfg5(n=64, batch=2)
    noisy = make_gpu(wn)
    with pytest.raises(phx.PhxError) as e:
        noisy.step_adaptive(0.1, 1e-8, 1e-6, 0.01)
    assert e.value.status == phx.PHX_ERR_UNSUPPORTED
    noisy.destroy()


def test_4096_grid_runs_on_device_without_host_round_trips():
    """Full-size smoke of the loop: 4096^2 fp32, a handful of attempts, finite fields, t advanced; one graph launch."""
    w = wl.cfg2(n=4096, prec="c32")
    g = make_gpu(w)
    before = g.get_launch_count()
    g.step_adaptive(0.05, 1e-6, 1e-4, 0.004, max_attempts=12)
    assert g.get_launch_count() == before + 1
    st = g.get_adaptive_state()
    assert 1 <= st["attempts"] <= 12 and st["t"] > 0 and st["n_accept"] >= 1
    assert np.all(np.isfinite(g.read_field("psi_p")[0, ::64]))
    g.destroy()
