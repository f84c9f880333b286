"""Pins of the CPU oracle against what the paper and the mathematics fix (all CPU, -m "not gpu").

None of these re-types the oracle's loops: each compares it with a closed form, a brute-force
definition, a 0-dimensional reduction integrated by an independent Python RK4 written from
Eqs. (2)-(6), (16), (17), or an invariant.  A dropped term, wrong sign, wrong index or swapped
operand anywhere in oracle/phx_oracle.cpp fails at least one of them.
"""
import numpy as np
import pytest

import oracle as orc


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def R4(z):
    """RK4 stability polynomial: one step of y' = lambda y multiplies y by R(lambda dt)."""
    return 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24


def plane_wave(nx, ny, p, q, batch=1):
    i = np.arange(nx)[None, :]
    j = np.arange(ny)[:, None]
    w = np.exp(1j * (2 * np.pi * p * i / nx + 2 * np.pi * q * j / ny))
    return np.broadcast_to(w, (batch, ny, nx)).copy()


# ----------------------------------------------------------------------------------------------
# Stencil, Eq. (8)
# ----------------------------------------------------------------------------------------------
def dense_laplacian(nx, ny, dx, dy, bc=(0, 0)):
    """Dense (nx*ny)^2 matrix straight from Eq. (8) with modular (or dropped) neighbour indices."""
    N = nx * ny
    A = np.zeros((N, N))
    for j in range(ny):
        for i in range(nx):
            k = j * nx + i
            for di, dj, w in ((1, 0, 1 / dx ** 2), (-1, 0, 1 / dx ** 2), (0, 1, 1 / dy ** 2), (0, -1, 1 / dy ** 2)):
                ii, jj = i + di, j + dj
                if bc[0] and not (0 <= ii < nx):
                    pass
                elif bc[1] and not (0 <= jj < ny):
                    pass
                else:
                    A[k, (jj % ny) * nx + (ii % nx)] += w
            A[k, k] += -2 / dx ** 2 - 2 / dy ** 2
    return A


@pytest.mark.parametrize("nx,ny,dx,dy,bc", [(8, 8, 0.5, 0.5, (0, 0)), (5, 7, 0.3, 0.7, (0, 0)),
                                             (7, 5, 0.3, 0.7, (1, 1)), (6, 4, 0.4, 0.9, (1, 0)),
                                             (3, 3, 1.0, 2.0, (0, 0))])
def test_stencil_vs_dense_bruteforce(nx, ny, dx, dy, bc):
    rng = np.random.default_rng(10)
    psi = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    # hbar = 1, m = 0.5  =>  hbar/2m = 1, K = i * Laplacian(psi)
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(hbar=1.0, m=0.5, dt=0.1), bc=bc)
    o.set_field("psi_p", psi)
    K = o.derivative()["K_p"]
    lap = (dense_laplacian(nx, ny, dx, dy, bc) @ psi.ravel()).reshape(ny, nx)
    assert rel_l2(K, 1j * lap) < 1e-14


def test_stencil_vs_fourier_symbol():
    nx, ny, dx, dy = 16, 12, 0.25, 0.4
    rng = np.random.default_rng(11)
    psi = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(hbar=2.0, m=0.25, dt=0.1))   # hbar/2m = 4
    o.set_field("psi_p", psi)
    K = o.derivative()["K_p"]
    a = 2 * np.pi * np.fft.fftfreq(nx)[None, :]
    b = 2 * np.pi * np.fft.fftfreq(ny)[:, None]
    k2 = (4 / dx ** 2) * np.sin(a / 2) ** 2 + (4 / dy ** 2) * np.sin(b / 2) ** 2
    lap = np.fft.ifft2(-k2 * np.fft.fft2(psi))
    assert rel_l2(K, 1j * 4.0 * lap) < 1e-13


# ----------------------------------------------------------------------------------------------
# TE-TM operator J_pm = Delta_LT (d_x -+ i d_y)^2 on the other component, compact
# nine-point form of DESIGN.md reading Q6, under periodic, zero and MIXED boundaries.
# The reference is a dense matrix assembled from 1-D shift matrices by Kronecker products: a value
# outside the grid along a zero axis is dropped, a periodic axis wraps.  (The 0-D plane-wave pin
# below is periodic-only; this one fixes the corner rule of the mixed case.)
# ----------------------------------------------------------------------------------------------
def shift_1d(n, d, zero_bc):
    """(S u)[i] = u[i + d] (d = +-1); outside the grid: 0 under a zero boundary, wrapped under a periodic one."""
    S = np.zeros((n, n))
    for i in range(n):
        k = i + d
        if 0 <= k < n:
            S[i, k] = 1.0
        elif not zero_bc:
            S[i, k % n] = 1.0
    return S


def dense_operators(nx, ny, dx, dy, bc):
    """d_xx, d_yy (three-point) and d_xy (product of the two central first differences) on the index k = j nx + i."""
    Ix, Iy = np.eye(nx), np.eye(ny)
    Xp, Xm = np.kron(Iy, shift_1d(nx, +1, bc[0])), np.kron(Iy, shift_1d(nx, -1, bc[0]))
    Yp, Ym = np.kron(shift_1d(ny, +1, bc[1]), Ix), np.kron(shift_1d(ny, -1, bc[1]), Ix)
    I = np.eye(nx * ny)
    dxx = (Xp + Xm - 2 * I) / dx ** 2
    dyy = (Yp + Ym - 2 * I) / dy ** 2
    dxy = ((Xp - Xm) / (2 * dx)) @ ((Yp - Ym) / (2 * dy))
    return dxx, dyy, dxy


@pytest.mark.parametrize("nx,ny,dx,dy,bc", [(6, 5, 0.5, 0.5, (1, 1)), (7, 4, 0.3, 0.7, (1, 0)), (6, 5, 0.4, 0.9, (0, 1)),
                                             (4, 7, 0.6, 0.35, (1, 0)), (3, 3, 0.5, 0.8, (0, 1)), (5, 6, 0.3, 0.45, (0, 0))])
def test_tetm_operator_vs_dense_bruteforce(nx, ny, dx, dy, bc):
    rng = np.random.default_rng(19)
    a = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    b = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    hbar, m, beta = 0.8, 0.4, 0.13
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(hbar=hbar, m=m, beta=beta, dt=0.1), model="spinor", bc=bc)
    o.set_field("psi_p", a)
    o.set_field("psi_m", b)
    K = o.derivative()
    dxx, dyy, dxy = dense_operators(nx, ny, dx, dy, bc)
    lap = dxx + dyy
    # Eq. (16): i hbar d_t psi_+- = -(hbar^2/2m) lap psi_+- + J_+- psi_-+,  J_+- = beta (d_x -+ i d_y)^2
    Jp = beta * (dxx - dyy - 2j * dxy)          # (d_x - i d_y)^2 acts on psi_- in the psi_+ equation
    Jm = beta * (dxx - dyy + 2j * dxy)
    Kp = (-1j / hbar) * (-(hbar ** 2) / (2 * m) * (lap @ a.ravel()) + Jp @ b.ravel())
    Km = (-1j / hbar) * (-(hbar ** 2) / (2 * m) * (lap @ b.ravel()) + Jm @ a.ravel())
    assert rel_l2(K["K_p"].ravel(), Kp) < 1e-13
    assert rel_l2(K["K_m"].ravel(), Km) < 1e-13
    # the coupling alone (no kinetic term would hide a wrong corner: compare K minus the Laplacian part too)
    assert rel_l2(K["K_p"].ravel() - 1j * hbar / (2 * m) * (lap @ a.ravel()), (-1j / hbar) * (Jp @ b.ravel())) < 1e-12


# ----------------------------------------------------------------------------------------------
# Linear scalar step: plane waves are exact eigenmodes, amplitude multiplies by R(z) per step
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("p,q", [(0, 0), (3, 0), (0, 5), (2, -3), (8, 8)])
def test_plane_wave_amplification(p, q):
    nx, ny, dx, dy = 16, 16, 0.5, 0.25
    hbar, m, V0, gamma, dt, N = 1.3, 0.7, 0.37, 0.05, 0.004, 25
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(hbar=hbar, m=m, gamma_c=gamma, dt=dt),
                   V=np.full((ny, nx), V0))
    psi0 = (0.3 - 0.2j) * plane_wave(nx, ny, p, q)
    o.set_field("psi_p", psi0)
    o.step_rk4(N)
    k2 = (4 / dx ** 2) * np.sin(np.pi * p / nx) ** 2 + (4 / dy ** 2) * np.sin(np.pi * q / ny) ** 2
    z = dt * (-1j * ((hbar / (2 * m)) * k2 + V0 / hbar) - gamma / 2)
    assert rel_l2(o.psi_p, R4(z) ** N * psi0) < 1e-13


def test_uniform_loss_closed_form():
    # V = g = 0, uniform field: |psi|^2 multiplies by R(-gamma dt/2)^2 per step exactly
    o = orc.Oracle(8, 8, 1.0, 1.0, orc.make_params(gamma_c=0.3, dt=0.05))
    o.set_field("psi_p", np.full((1, 8, 8), 0.8 + 0.1j))
    n0 = np.abs(o.psi_p) ** 2
    o.step_rk4(40)
    assert rel_l2(np.abs(o.psi_p) ** 2, n0 * R4(-0.3 * 0.05 / 2) ** 80) < 1e-13


def test_norm_drift_of_linear_lossless_step():
    # gamma = 0: |R(i theta)|^2 = 1 - theta^6/72 + theta^8/576 for every mode
    nx = ny = 8
    dx, dt = 0.5, 0.02
    o = orc.Oracle(nx, ny, dx, dx, orc.make_params(dt=dt))
    o.set_field("psi_p", plane_wave(nx, ny, 2, 1))
    o.step_rk4(1)
    theta = dt * ((4 / dx ** 2) * (np.sin(np.pi * 2 / nx) ** 2 + np.sin(np.pi * 1 / ny) ** 2))
    expect = 1 - theta ** 6 / 72 + theta ** 8 / 576
    assert abs(np.mean(np.abs(o.psi_p) ** 2) - expect) < 1e-14


def test_zero_boundary_sine_modes():
    # zero (Dirichlet) boundaries: sin modes are the eigenmodes of the stencil
    nx, ny, dx, dy, dt, N = 9, 6, 0.5, 0.4, 0.01, 10
    p, q = 2, 3
    i = np.arange(nx)[None, :] + 1
    j = np.arange(ny)[:, None] + 1
    mode = np.sin(np.pi * p * i / (nx + 1)) * np.sin(np.pi * q * j / (ny + 1)) * (1 + 0.5j)
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(gamma_c=0.1, dt=dt), bc=(1, 1))
    o.set_field("psi_p", mode)
    o.step_rk4(N)
    k2 = (4 / dx ** 2) * np.sin(np.pi * p / (2 * (nx + 1))) ** 2 + (4 / dy ** 2) * np.sin(np.pi * q / (2 * (ny + 1))) ** 2
    z = dt * (-1j * k2 - 0.05)
    assert rel_l2(o.psi_p[0], R4(z) ** N * mode) < 1e-13


# ----------------------------------------------------------------------------------------------
# 0-dimensional reduction: a plane wave with uniform V, P, n stays a plane wave under the
# discrete RK4 map, so the grid result equals an RK4 on the amplitudes with the stencils replaced
# by their symbols.  The reference below is written from Eqs. (2)-(6), (16), (17) in physical
# parameters (not from the oracle's coefficient set).
# ----------------------------------------------------------------------------------------------
def rk4_0d(f, u, t, dt):
    k1 = f(t, u)
    k2 = f(t + dt / 2, u + 0.5 * dt * k1)
    k3 = f(t + dt / 2, u + 0.5 * dt * k2)
    k4 = f(t + dt, u + dt * k3)
    return u + (dt / 6) * k1 + (dt / 3) * k2 + (dt / 3) * k3 + (dt / 6) * k4


def rhs_0d(prm, dx, dy, a, b, V0, P0, E0, spinor, reservoir):
    """State u = [A+, A-, n+, n-] (complex array); a, b = phase advance per cell in x, y."""
    hb, m = prm["hbar"], prm["m"]
    dxx = -(4 / dx ** 2) * np.sin(a / 2) ** 2           # symbol of d_xx (three-point)
    dyy = -(4 / dy ** 2) * np.sin(b / 2) ** 2
    dxy = -np.sin(a) * np.sin(b) / (dx * dy)            # symbol of d_xy (four-corner)

    def f(t, u):
        A = [u[0], u[1]]
        n = [u[2].real, u[3].real]
        out = np.zeros(4, dtype=complex)
        for s in range(2 if spinor else 1):
            o = 1 - s
            rho = abs(A[s]) ** 2 - prm.get("density_offset", 0.0)
            rho_o = abs(A[o]) ** 2 - prm.get("density_offset", 0.0) if spinor else 0.0
            nn = n[s] if reservoir else 0.0
            H = (-(hb ** 2) / (2 * m) * (dxx + dyy) + V0 + prm.get("g", 0) * rho + prm.get("g_x", 0) * rho_o
                 + prm.get("g_r", 0) * nn + 0.5j * hb * (prm.get("R", 0) * nn - prm.get("gamma_c", 0)))
            dA = -1j / hb * H * A[s]
            if spinor:
                sgn = -1 if s == 0 else +1                # (d_x -+ i d_y)^2 = d_xx - d_yy -+ 2i d_xy
                J = prm.get("beta", 0) * (dxx - dyy + sgn * 2j * dxy)
                dA += -1j / hb * J * A[o]
            dA += -1j / hb * E0 * np.exp(-1j * prm.get("omega", 0.0) * t)
            out[s] = dA
            if reservoir:
                out[2 + s] = P0 - (prm.get("gamma_r", 0) + prm.get("R", 0) * rho) * nn
        return out
    return f


CASES_0D = [
    ("scalar", dict(hbar=1.0, m=0.5, g=1.0, gamma_c=0.01, dt=0.01), 0.4, 0.0, 0.0),
    ("scalar", dict(hbar=0.8, m=0.3, g=-0.7, gamma_c=0.2, dt=0.004, density_offset=0.05), -0.3, 0.0, 0.0),
    ("reservoir", dict(hbar=0.6582, m=0.57, g=0.3, g_r=0.6, R=0.4, gamma_c=0.15, gamma_r=0.225, dt=0.01),
     0.1, 2.0, 0.0),
    ("spinor", dict(hbar=1.0, m=0.5, g=0.5, g_x=-0.2, beta=0.1, gamma_c=0.05, dt=0.004), 0.0, 0.0, 0.0),
    ("spinor_reservoir", dict(hbar=0.9, m=0.4, g=0.5, g_x=0.1, g_r=0.3, R=0.2, beta=0.07, gamma_c=0.1,
                              gamma_r=0.3, dt=0.005), 0.2, 1.5, 0.0),
    ("scalar", dict(hbar=1.0, m=0.5, g=0.3, gamma_c=0.1, dt=0.01, omega=1.7), 0.0, 0.0, 0.25 - 0.1j),
    ("spinor_reservoir", dict(hbar=0.9, m=0.4, g=0.5, g_x=0.1, g_r=0.3, R=0.2, beta=0.07, gamma_c=0.1,
                              gamma_r=0.3, dt=0.005, omega=-0.6), 0.2, 1.5, 0.1 + 0.3j),
]


@pytest.mark.parametrize("model,prm,V0,P0,E0", CASES_0D)
@pytest.mark.parametrize("p,q", [(0, 0), (1, 2), (-3, 1)])
def test_zero_dimensional_reduction(model, prm, V0, P0, E0, p, q):
    nx, ny, dx, dy, N = 12, 10, 0.5, 0.35, 30
    spinor = model.startswith("spinor")
    reservoir = model.endswith("reservoir")
    wave = plane_wave(nx, ny, p, q)
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(**prm), model=model, V=np.full((ny, nx), V0),
                   P=np.full((ny, nx), P0) if reservoir else None,
                   E=(E0 * wave[0]) if E0 != 0 else None)
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
    dt = prm["dt"]
    for s in range(N):
        u = rk4_0d(f, u, s * dt, dt)
    o.step_rk4(N)
    assert rel_l2(o.psi_p, u[0] * wave) < 1e-12
    if spinor:
        assert rel_l2(o.psi_m, u[1] * wave) < 1e-12
    if reservoir:
        assert rel_l2(o.n_p, np.full((1, ny, nx), u[2].real)) < 1e-12
        if spinor:
            assert rel_l2(o.n_m, np.full((1, ny, nx), u[3].real)) < 1e-12


def test_reservoir_alone_closed_form():
    # psi = 0: dn/dt = P - gamma_r n  =>  n_N = R(z)^N n0 + (P/gamma_r)(1 - R(z)^N), z = -gamma_r dt
    nx = ny = 6
    rng = np.random.default_rng(12)
    P = rng.uniform(0.5, 2.0, (ny, nx))
    n0 = rng.uniform(0.0, 3.0, (1, ny, nx))
    gr, dt, N = 0.225, 0.05, 60
    o = orc.Oracle(nx, ny, 1.0, 1.0, orc.make_params(R=0.01, g_r=0.2, gamma_c=0.15, gamma_r=gr, dt=dt),
                   model="reservoir", P=P)
    o.set_field("n_p", n0)
    o.step_rk4(N)
    rz = R4(-gr * dt) ** N
    assert rel_l2(o.n_p, rz * n0 + (P / gr) * (1 - rz)) < 1e-13
    assert np.all(o.psi_p == 0)


# ----------------------------------------------------------------------------------------------
# Reductions between models, invariances, order of accuracy
# ----------------------------------------------------------------------------------------------
def _random_state(rng, shape, amp=0.5):
    return amp * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))


def test_spinor_without_coupling_is_two_scalars():
    nx, ny = 10, 7
    rng = np.random.default_rng(13)
    V = rng.standard_normal((ny, nx)) * 0.1
    prm = dict(g=0.8, gamma_c=0.1, dt=0.01)
    a, b = _random_state(rng, (1, ny, nx)), _random_state(rng, (1, ny, nx))
    sp = orc.Oracle(nx, ny, 0.5, 0.6, orc.make_params(**prm), model="spinor", V=V)
    sp.set_field("psi_p", a)
    sp.set_field("psi_m", b)
    sp.step_rk4(20)
    for init, got in ((a, sp.psi_p), (b, sp.psi_m)):
        sc = orc.Oracle(nx, ny, 0.5, 0.6, orc.make_params(**prm), V=V)
        sc.set_field("psi_p", init)
        sc.step_rk4(20)
        assert np.array_equal(sc.psi_p, got)


def test_reservoir_decoupled_is_scalar():
    nx, ny = 9, 8
    rng = np.random.default_rng(14)
    a = _random_state(rng, (1, ny, nx))
    prm = dict(g=0.8, gamma_c=0.1, dt=0.01)
    rs = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(gamma_r=0.2, **prm), model="reservoir",
                    P=np.ones((ny, nx)))
    rs.set_field("psi_p", a)
    rs.step_rk4(15)
    sc = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(**prm))
    sc.set_field("psi_p", a)
    sc.step_rk4(15)
    assert np.array_equal(sc.psi_p, rs.psi_p)


def test_shift_equivariance_and_step_splitting():
    nx, ny = 11, 9
    rng = np.random.default_rng(15)
    V = rng.standard_normal((ny, nx)) * 0.2
    P = rng.uniform(0, 2, (ny, nx))
    prm = orc.make_params(g=0.5, g_x=0.2, g_r=0.3, R=0.1, gamma_c=0.1, gamma_r=0.2, beta=0.05, dt=0.01)
    st = {k: _random_state(rng, (1, ny, nx)) for k in ("psi_p", "psi_m")}
    st["n_p"] = rng.uniform(0, 1, (1, ny, nx))
    st["n_m"] = rng.uniform(0, 1, (1, ny, nx))

    def run(shift, split):
        o = orc.Oracle(nx, ny, 0.5, 0.4, prm, model="spinor_reservoir", V=np.roll(V, shift, (0, 1)),
                       P=np.roll(P, shift, (0, 1)))
        for k, v in st.items():
            o.set_field(k, np.roll(v, shift, (1, 2)))
        for n in split:
            o.step_rk4(n)
        return o
    base = run((0, 0), [12])
    moved = run((4, -3), [5, 7])
    for k in st:
        assert np.array_equal(np.roll(getattr(base, k), (4, -3), (1, 2)), getattr(moved, k))


def test_rk4_is_fourth_order():
    nx = ny = 12
    rng = np.random.default_rng(16)
    psi0 = _random_state(rng, (1, ny, nx), 0.4)
    V = 0.3 * rng.standard_normal((ny, nx))

    def run(dt, n):
        o = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(g=1.0, gamma_c=0.05, dt=dt), V=V)
        o.set_field("psi_p", psi0)
        o.step_rk4(n)
        return o.psi_p
    ref = run(0.04 / 32, 10 * 32)
    e1 = rel_l2(run(0.04, 10), ref)
    e2 = rel_l2(run(0.02, 20), ref)
    assert 13.0 < e1 / e2 < 19.0


def test_gauge_factor_i_commutes_with_scalar_step():
    # psi -> i psi is an exact symmetry of Eq. (1); multiplying by i is exact in floating point
    nx, ny = 8, 8
    rng = np.random.default_rng(17)
    a = _random_state(rng, (1, ny, nx))
    outs = []
    for fac in (1, 1j):
        o = orc.Oracle(nx, ny, 0.5, 0.5, orc.make_params(g=0.9, gamma_c=0.1, dt=0.01))
        o.set_field("psi_p", fac * a)
        o.step_rk4(10)
        outs.append(o.psi_p)
    assert np.array_equal(1j * outs[0], outs[1])


def test_canonical_coefficients():
    prm = orc.make_params(hbar=6.582e-4, m=5.7e-4, g=6e-6, g_r=12e-6, R=0.01, gamma_c=0.15, gamma_r=0.225,
                          beta=0.1, dt=1e-3, noise_scale=2.0, density_offset=0.5)
    dx, dy = 200 / 4096, 0.07
    c = dict(zip(orc.COEF_NAMES, orc.derive_coeffs(prm, dx, dy, False)))
    assert c["cx"] == 6.582e-4 / (2 * 5.7e-4 * dx * dx) and c["cy"] == 6.582e-4 / (2 * 5.7e-4 * dy * dy)
    assert c["ih"] == 1 / 6.582e-4 and c["hgc"] == 0.075 and c["gamr"] == 0.225 and c["Rr"] == 0.01
    assert c["bxx"] == 0.1 / (6.582e-4 * dx * dx) and c["byy"] == 0.1 / (6.582e-4 * dy * dy)
    assert c["bxy"] == 0.1 / (2 * 6.582e-4 * dx * dy)
    assert c["dt6"] == 1e-3 / 6 and c["dt3"] == 1e-3 / 3 and c["sig2"] == 2.0 * 1e-3 / (4 * dx * dy)
    c32 = orc.derive_coeffs(prm, dx, dy, True)
    assert np.array_equal(c32, c32.astype(np.float32).astype(np.float64))
    assert np.allclose(c32, list(c.values()), rtol=1e-7)


def test_batch_elements_are_independent_runs():
    nx, ny, B = 6, 5, 3
    rng = np.random.default_rng(18)
    a = _random_state(rng, (B, ny, nx))
    prm = orc.make_params(g=0.5, gamma_c=0.1, dt=0.02)
    ob = orc.Oracle(nx, ny, 0.5, 0.5, prm, batch=B)
    ob.set_field("psi_p", a)
    ob.step_rk4(7)
    for r in range(B):
        o1 = orc.Oracle(nx, ny, 0.5, 0.5, prm)
        o1.set_field("psi_p", a[r:r + 1])
        o1.step_rk4(7)
        assert np.array_equal(o1.psi_p[0], ob.psi_p[r])
