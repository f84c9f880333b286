"""Pins of the oracle's adaptive Dormand-Prince 5(4) integrator (the paper names the method at
PAPER.md:64 and :488 and gives nothing else, so every rule is DESIGN.md reading Q20).  All CPU, -m "not gpu".

What fixes it, independently of the oracle's own loops:
  - the tableau against the ORDER CONDITIONS (rooted trees up to order 5 for b, order 4 for b* = b - e), the row sums and
    the known sixth coefficient 1/600 of the stability polynomial -- a wrong digit in any coefficient fails one;
  - a linear plane wave: one step multiplies the amplitude by R(z) = sum_{k<=5} z^k/k! + z^6/600 exactly;
  - fifth-order convergence of the fixed-step solution and h^5 scaling of the error estimate on a nonlinear grid problem;
  - the whole controller (error norm, accept rule, quantised factor, clamp, clipping at t_end, FSAL) against an independent
    0-dimensional Dormand-Prince integrator written here from the published coefficients as exact fractions, on plane-wave
    states (which stay plane waves, so the grid's max-norm equals the 0-D value): accept / q sequences equal as integers;
  - interrupting a run (max_attempts) and resuming it changes nothing, bit for bit."""
from fractions import Fraction as Fr

import numpy as np
import pytest

import oracle as orc
from test_oracle_pins import plane_wave, rel_l2, rhs_0d


# ---- the tableau ------------------------------------------------------------------------------------------------
def test_tableau_row_sums_and_order_conditions():
    c, A, b, e = orc.dp54_tableau()
    bs = b - e                                                   # embedded fourth-order weights
    one = np.ones(7)
    assert np.allclose(A.sum(1), c, atol=3e-16)
    assert np.all(np.triu(A) == 0)                               # explicit
    assert np.array_equal(A[6], b)                               # FSAL: the last stage is evaluated at u_new
    C = np.diag(c)
    # all 17 rooted trees up to order 5: elementary weight Phi(tree) and density gamma(tree); sum b_i Phi_i = 1/gamma
    Ac, Ac2, Ac3 = A @ c, A @ c ** 2, A @ c ** 3
    trees = [
        (one, 1), (c, 2), (c ** 2, 3), (Ac, 6),
        (c ** 3, 4), (c * Ac, 8), (Ac2, 12), (A @ Ac, 24),
        (c ** 4, 5), (c ** 2 * Ac, 10), (c * Ac2, 15), (c * (A @ Ac), 30), (Ac * Ac, 20),
        (Ac3, 20), (A @ (c * Ac), 40), (A @ Ac2, 60), (A @ (A @ Ac), 120),
    ]
    for k, (phi, gamma) in enumerate(trees):
        assert abs(b @ phi - 1.0 / gamma) < 5e-16, f"order condition {k} of b"
    for k, (phi, gamma) in enumerate(trees[:8]):                 # b* is fourth order
        assert abs(bs @ phi - 1.0 / gamma) < 5e-16, f"order condition {k} of b*"
    assert abs(bs @ (c ** 4) - 0.2) > 1e-4                        # ... and not fifth
    # stability polynomial: b A^k 1 = 1/(k+1)! for k <= 4 and the known 1/600 for k = 5
    v = one.copy()
    coef = []
    for k in range(6):
        coef.append(b @ v)
        v = A @ v
    assert np.allclose(coef, [1, 1 / 2, 1 / 6, 1 / 24, 1 / 120, 1 / 600], atol=3e-16)
    c32, A32, b32, e32 = orc.dp54_tableau(prec32=True)
    for x, y in ((c32, c), (A32, A), (b32, b), (e32, e)):
        assert np.array_equal(x, x.astype(np.float32).astype(np.float64)) and np.allclose(x, y, rtol=1e-7, atol=0)


def R_dp5(z):
    return 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24 + z ** 5 / 120 + z ** 6 / 600


def _fixed(h):
    """Controller settings that force a constant step h (h_min = h_max: a step that cannot shrink is accepted)."""
    return dict(atol=1e-30, rtol=1e-30, h_init=h, h_min=h, h_max=h)


@pytest.mark.parametrize("p,q", [(0, 0), (3, 1), (2, -5)])
def test_plane_wave_amplification_is_the_stability_polynomial(p, q):
    nx, ny, dx, dy = 16, 12, 0.5, 0.25
    hbar, m, V0, gamma, h, N = 1.3, 0.7, 0.37, 0.05, 0.01, 8
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(hbar=hbar, m=m, gamma_c=gamma, dt=1.0), V=np.full((ny, nx), V0))
    psi0 = (0.3 - 0.2j) * plane_wave(nx, ny, p, q)
    o.set_field("psi_p", psi0)
    log = o.step_dp54(N * h, **_fixed(h))
    assert log["attempts"] == N and np.all(log["accept"] == 1)
    k2 = (4 / dx ** 2) * np.sin(np.pi * p / nx) ** 2 + (4 / dy ** 2) * np.sin(np.pi * q / ny) ** 2
    z = h * (-1j * ((hbar / (2 * m)) * k2 + V0 / hbar) - gamma / 2)
    assert rel_l2(o.psi_p, R_dp5(z) ** N * psi0) < 1e-13


def _nonlinear_problem(model="scalar"):
    nx = ny = 12
    rng = np.random.default_rng(21)
    st = {"psi_p": 0.4 * (rng.standard_normal((1, ny, nx)) + 1j * rng.standard_normal((1, ny, nx)))}
    prm = dict(g=1.0, gamma_c=0.05)
    kw = dict(V=0.3 * rng.standard_normal((ny, nx)))
    if model == "spinor_reservoir":
        st["psi_m"] = 0.4 * (rng.standard_normal((1, ny, nx)) + 1j * rng.standard_normal((1, ny, nx)))
        st["n_p"] = rng.uniform(0, 1, (1, ny, nx))
        st["n_m"] = rng.uniform(0, 1, (1, ny, nx))
        prm.update(g_x=0.3, g_r=0.4, R=0.2, gamma_r=0.3, beta=0.05)
        kw["P"] = rng.uniform(0, 2, (ny, nx))

    def make(dt=1.0):
        o = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(dt=dt, **prm), model=model, **kw)
        for k, v in st.items():
            o.set_field(k, v)
        return o
    return make, list(st)


@pytest.mark.parametrize("model", ["scalar", "spinor_reservoir"])
def test_fixed_step_solution_is_fifth_order_and_error_estimate_scales_as_h5(model):
    make, names = _nonlinear_problem(model)
    T = 0.32
    ref = make(dt=T / 2560)
    ref.step_rk4(2560)                                           # fine RK4 reference (error ~ 1e-13)
    errs, ests = [], []
    for n in (8, 16):
        o = make()
        log = o.step_dp54(T, **_fixed(T / n))
        assert log["attempts"] == n
        errs.append(max(rel_l2(getattr(o, k), getattr(ref, k)) for k in names))
        ests.append(log["err"][0])
    assert 24.0 < errs[0] / errs[1] < 40.0, errs                 # global error ~ h^5
    assert 24.0 < ests[0] / ests[1] < 40.0, ests                 # E = u_5 - u_4 ~ h^5 per step


# ---- the controller against an independent 0-dimensional integrator ---------------------------------------------------
A_FR = [[], [Fr(1, 5)], [Fr(3, 40), Fr(9, 40)], [Fr(44, 45), Fr(-56, 15), Fr(32, 9)],
        [Fr(19372, 6561), Fr(-25360, 2187), Fr(64448, 6561), Fr(-212, 729)],
        [Fr(9017, 3168), Fr(-355, 33), Fr(46732, 5247), Fr(49, 176), Fr(-5103, 18656)],
        [Fr(35, 384), Fr(0), Fr(500, 1113), Fr(125, 192), Fr(-2187, 6784), Fr(11, 84)]]
BSTAR_FR = [Fr(5179, 57600), Fr(0), Fr(7571, 16695), Fr(393, 640), Fr(-92097, 339200), Fr(187, 2100), Fr(1, 40)]


def dp54_0d(f, u, t, t_end, atol, rtol, h, h_min, h_max, absval):
    """Adaptive Dormand-Prince 5(4) on a small state vector, every rule of DESIGN.md reading Q20 written out again."""
    a = [[float(x) for x in row] for row in A_FR]
    c = [sum(row) for row in a]
    b = a[6] + [0.0]
    e = [b[j] - float(BSTAR_FR[j]) for j in range(7)]
    log = []
    k1 = None
    while t < t_end:
        clipped = t + h >= t_end
        hu = t_end - t if clipped else h
        K = [f(t, u) if k1 is None else k1]
        for s in range(1, 7):
            y = u + hu * sum(a[s][j] * K[j] for j in range(s))
            K.append(f(t + c[s] * hu, y))
        un = u + hu * sum(b[j] * K[j] for j in range(6))
        E = hu * sum(e[j] * K[j] for j in range(7))
        err = max(absval(E) / (atol + rtol * np.maximum(absval(u), absval(un))))
        accept = err <= 1.0 or h <= h_min
        fac = min(4.0, max(0.25, 0.9 * err ** -0.2)) if err > 0 else 4.0
        q = int(np.floor(16.0 * fac))
        log.append((int(accept), q, hu, err))
        if accept:
            u, k1 = un, K[6]
            t = t_end if clipped else t + hu
            if not clipped:
                h = min(h_max, max(h_min, hu * q / 16.0))
        else:
            h = min(h_max, max(h_min, hu * q / 16.0))
    return u, h, log


CASES = [
    ("scalar", dict(hbar=1.0, m=0.5, g=1.0, gamma_c=0.01), 0.4, 0.0, 0.0),
    ("reservoir", dict(hbar=0.6582, m=0.57, g=0.3, g_r=0.6, R=0.4, gamma_c=0.15, gamma_r=0.225), 0.1, 2.0, 0.0),
    ("spinor_reservoir", dict(hbar=0.9, m=0.4, g=0.5, g_x=0.1, g_r=0.3, R=0.2, beta=0.07, gamma_c=0.1, gamma_r=0.3, omega=-0.6),
     0.2, 1.5, 0.1 + 0.3j),
]


@pytest.mark.parametrize("model,prm,V0,P0,E0", CASES)
@pytest.mark.parametrize("tol", [(1e-7, 1e-5), (1e-10, 1e-8)])
def test_controller_against_zero_dimensional_integrator(model, prm, V0, P0, E0, tol):
    nx, ny, dx, dy, p, q = 12, 10, 0.5, 0.35, 1, 2
    spinor, reservoir = model.startswith("spinor"), model.endswith("reservoir")
    wave = plane_wave(nx, ny, p, q)
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(dt=1.0, **prm), model=model, V=np.full((ny, nx), V0),
                   P=np.full((ny, nx), P0) if reservoir else None, E=(E0 * wave[0]) if E0 != 0 else None)
    u = np.array([0.7 - 0.2j, (0.1 + 0.5j) if spinor else 0, 0.3 if reservoir else 0, 0.9 if reservoir and spinor else 0],
                 dtype=complex)
    o.set_field("psi_p", u[0] * wave)
    if spinor:
        o.set_field("psi_m", u[1] * wave)
    if reservoir:
        o.set_field("n_p", np.full((1, ny, nx), u[2].real))
        if spinor:
            o.set_field("n_m", np.full((1, ny, nx), u[3].real))
    f = rhs_0d(prm, dx, dy, 2 * np.pi * p / nx, 2 * np.pi * q / ny, V0, P0, E0, spinor, reservoir)
    atol, rtol = tol
    t_end, h0, h_min, h_max = 1.3, 0.2, 1e-6, 0.09                  # h0 > h_max: clamped; several rejections at the start
    log = o.step_dp54(t_end, atol, rtol, h0, h_min, h_max)
    u_ref, h_ref, log_ref = dp54_0d(f, u, 0.0, t_end, atol, rtol, min(h0, h_max), h_min, h_max, np.abs)
    # the decisions are integers: they agree exactly unless err sits within rounding of a decision boundary
    margin = min(min(abs(r[3] - 1.0), abs(16 * 0.9 * r[3] ** -0.2 % 1.0), abs(1 - 16 * 0.9 * r[3] ** -0.2 % 1.0)) for r in log_ref)
    assert margin > 1e-9, "test case sits on a decision boundary: choose other parameters"
    assert log["attempts"] == len(log_ref)
    assert np.array_equal(log["accept"], [r[0] for r in log_ref])
    assert np.array_equal(log["q"], [r[1] for r in log_ref])
    assert np.allclose(log["h"], [r[2] for r in log_ref], rtol=1e-14, atol=0)
    assert np.allclose(log["err"], [r[3] for r in log_ref], rtol=1e-8)
    assert (log["accept"] == 0).sum() >= 1 and o.ad.n_reject == (log["accept"] == 0).sum()
    assert o.ad.t == t_end and abs(o.ad.h_next - h_ref) <= 1e-14 * h_ref
    assert rel_l2(o.psi_p, u_ref[0] * wave) < 1e-12
    if spinor:
        assert rel_l2(o.psi_m, u_ref[1] * wave) < 1e-12
    if reservoir:
        assert rel_l2(o.n_p, np.full((1, ny, nx), u_ref[2].real)) < 1e-12


def test_tolerance_controls_the_global_error():
    make, names = _nonlinear_problem("scalar")
    T = 0.5
    ref = make(dt=T / 4000)
    ref.step_rk4(4000)
    errs = []
    for rtol in (1e-4, 1e-6, 1e-8):
        o = make()
        o.step_dp54(T, atol=rtol * 1e-2, rtol=rtol, h_init=0.05, h_max=0.2)
        errs.append(rel_l2(o.psi_p, ref.psi_p))
    assert errs[0] > errs[1] > errs[2] and errs[0] < 1e-3 and errs[2] < 1e-7, errs


def test_interrupted_run_resumes_bit_for_bit_and_batch_shares_one_step_size():
    make, names = _nonlinear_problem("spinor_reservoir")
    a = make()
    log_a = a.step_dp54(0.4, 1e-9, 1e-7, 0.05)
    b = make()
    log_b1 = b.step_dp54(0.4, 1e-9, 1e-7, 0.05, max_attempts=5)
    assert log_b1["attempts"] == 5 and b.ad.t < 0.4
    log_b2 = b.step_dp54(0.4, 1e-9, 1e-7, 0.05)
    assert b.ad.t == a.ad.t == 0.4 and b.ad.h_next == a.ad.h_next
    assert np.array_equal(np.concatenate([log_b1["q"], log_b2["q"]]), log_a["q"])
    for k in names:
        assert np.array_equal(getattr(a, k), getattr(b, k))
    # a batch of two different states takes the steps its stiffer element needs: same h sequence for both elements
    nx = ny = 12
    rng = np.random.default_rng(22)
    s0 = 0.4 * (rng.standard_normal((2, ny, nx)) + 1j * rng.standard_normal((2, ny, nx)))
    s0[1] *= 3.0
    ob = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(g=1.0, gamma_c=0.05, dt=1.0), batch=2)
    ob.set_field("psi_p", s0)
    lb = ob.step_dp54(0.3, 1e-9, 1e-7, 0.05)
    o1 = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(g=1.0, gamma_c=0.05, dt=1.0))
    o1.set_field("psi_p", s0[1:2])
    l1 = o1.step_dp54(0.3, 1e-9, 1e-7, 0.05)
    assert np.array_equal(lb["q"], l1["q"]) and np.array_equal(ob.psi_p[1], o1.psi_p[0])


def test_noise_is_refused():
    o = orc.Oracle(8, 8, 0.5, 0.5, orc.make_params(gamma_c=0.1, dt=0.01), noise=True, seed=1)
    with pytest.raises(RuntimeError):
        o.step_dp54(0.1, 1e-8, 1e-6, 0.01)
