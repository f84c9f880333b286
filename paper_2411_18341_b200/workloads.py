"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module holds NO arithmetic of the method (no stencil, no RK4, no Philox): it only draws the
initial fields, potentials and pumps with numpy and rounds them once to the working precision.
The same arrays are handed unchanged to the CUDA library and (in tests / bench cpu_baseline) to the
oracle.  The paper ships its inputs in its repository, which is not
available here; these arrays stand in for them.

Conventions (readings Q3, Q14): arrays are [batch][ny][nx], x fastest;
x_i = (i - nx/2) dx, y_j = (j - ny/2) dy; "complex normal of std s" has re, im ~ N(0, s^2/2).
"""
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

_CDT = {"c32": np.complex64, "c64": np.complex128}
_RDT = {"c32": np.float32, "c64": np.float64}


@dataclass
class Workload:
    name: str
    model: str                      # "scalar" | "reservoir" | "spinor" | "spinor_reservoir"
    prec: str                       # "c32" | "c64"
    nx: int
    ny: int
    batch: int
    dx: float
    dy: float
    params: dict                    # hbar, m, g, g_x, g_r, R, gamma_c, gamma_r, beta, dt, noise_scale, ...
    n_steps: int
    noise: bool = False
    seed: int = 0
    V: Optional[np.ndarray] = None  # [ny][nx] real T
    P: Optional[np.ndarray] = None  # [ny][nx] real T
    fields: dict = field(default_factory=dict)   # "psi_p", "psi_m", "n_p", "n_m" -> [batch][ny][nx]

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.batch


def _coords(nx, ny, dx, dy):
    x = (np.arange(nx) - nx // 2) * dx
    y = (np.arange(ny) - ny // 2) * dy
    return x[None, :], y[:, None]


def _cnormal(rng, shape, std, cdt):
    """Complex normal with E|z|^2 = std^2, drawn row-block-wise to bound float64 temporaries."""
    out = np.empty(shape, dtype=cdt)
    flat = out.reshape(-1)
    s = std / np.sqrt(2.0)
    blk = 1 << 22
    for a in range(0, flat.size, blk):
        b = min(flat.size, a + blk)
        flat[a:b] = (rng.standard_normal(b - a) * s + 1j * (rng.standard_normal(b - a) * s)).astype(cdt)
    return out


def ring_pump(nx, ny, dx, dy, P0, w, rdt):
    """Eq. (21) with the sign of the exponent fixed (reading Q10): P0 (r/w)^2 exp(-(r/w)^2)."""
    x, y = _coords(nx, ny, dx, dy)
    q = (x * x + y * y) / (w * w)
    return (P0 * q * np.exp(-q)).astype(rdt)


def smooth_disorder(nx, ny, corr_cells, std, rng, rdt):
    """Periodic Gaussian filter (sigma = corr_cells) of N(0,1) noise, mean removed, scaled to `std`."""
    white = rng.standard_normal((ny, nx))
    kx = np.fft.fftfreq(nx)[None, :] * 2 * np.pi
    ky = np.fft.fftfreq(ny)[:, None] * 2 * np.pi
    filt = np.exp(-0.5 * corr_cells ** 2 * (kx * kx + ky * ky))
    v = np.fft.ifft2(np.fft.fft2(white) * filt).real
    v -= v.mean()
    v *= std / v.std()
    return v.astype(rdt)


def cfg1(n=64, prec="c64", n_steps=1000):
    """Config 1: scalar Eq. (1), 64x64, harmonic V, Gaussian x plane wave + noise, complex fp64."""
    dx = 0.5
    cdt, rdt = _CDT[prec], _RDT[prec]
    rng = np.random.default_rng(0)
    x, y = _coords(n, n, dx, dx)
    r2 = x * x + y * y
    L = n * dx
    kx = 2 * np.pi * 3 / L
    psi = np.exp(-r2 / (2 * 4.0 ** 2)) * np.exp(1j * kx * x)
    psi = (psi + _cnormal(rng, (n, n), 1e-3, np.complex128)).astype(cdt)
    return Workload("cfg1", "scalar", prec, n, n, 1, dx, dx,
                    dict(hbar=1.0, m=0.5, g=1.0, gamma_c=0.01, dt=0.01), n_steps, V=(0.01 * r2).astype(rdt),
                    fields={"psi_p": psi[None]})


def cfg2(n=4096, prec="c32", n_steps=10000, ny=None, tile=None):
    """Config 2: scalar Eq. (1), n x n (1024, 4096), smooth disorder V, uniform random psi0.

    tile=t (t divides n, square grids): the recipe is drawn on a t x t grid and repeated periodically to n x n (the disorder is
    periodic, so the tiling is seamless); used by bench.py for sizes beyond BASELINE's (8192^2, 16384^2), ready in seconds."""
    if tile is not None and tile != n:
        if n % tile != 0 or ny not in (None, n):
            raise ValueError("tile must divide n (square grids)")
        w = cfg2(tile, prec, n_steps)
        reps = n // tile
        w.V = np.tile(w.V, (reps, reps))
        w.fields = {k: np.tile(v, (1, reps, reps)) for k, v in w.fields.items()}
        w.name, w.nx, w.ny = f"cfg2_{n}x{n}_{prec}", n, n
        return w
    dx = 0.2
    ny = n if ny is None else ny
    cdt, rdt = _CDT[prec], _RDT[prec]
    rng = np.random.default_rng(1)
    V = smooth_disorder(n, ny, 5.0, 0.05, rng, rdt)
    a = 0.1 / np.sqrt(2.0)
    psi = np.empty((1, ny, n), dtype=cdt)
    for j0 in range(0, ny, 256):
        j1 = min(ny, j0 + 256)
        psi[0, j0:j1] = (rng.uniform(-a, a, (j1 - j0, n)) + 1j * rng.uniform(-a, a, (j1 - j0, n))).astype(cdt)
    return Workload(f"cfg2_{n}x{ny}_{prec}", "scalar", prec, n, ny, 1, dx, dx,
                    dict(hbar=1.0, m=0.5, g=2e-3, gamma_c=0.1, dt=0.004), n_steps, V=V, fields={"psi_p": psi})


# Config 3 physics in consistent eV / ps / um units (reading Q9).
_POLARITON = dict(hbar=6.582e-4, m=5.7e-4, g=6e-6, g_r=12e-6, R=0.01, gamma_c=0.15, gamma_r=0.225)


def cfg3(n=4096, prec="c32", n_steps=50000, keep_dx=True):
    """Config 3: polariton condensate with reservoir, ring pump, 200 um box at n=4096.

    For n != 4096 with keep_dx the cell size of the full config is kept (box shrinks, ring radius
    stays 0.15 L) so that reduced parity cases have the same stiffness omega_max*dt = 1.94."""
    cdt, rdt = _CDT[prec], _RDT[prec]
    dx = 200.0 / 4096 if keep_dx else 200.0 / n
    L = n * dx
    rng = np.random.default_rng(2)
    psi = _cnormal(rng, (1, n, n), 1e-2, cdt)
    P = ring_pump(n, n, dx, dx, 100.0, 0.15 * L, rdt)
    prm = dict(_POLARITON, dt=1.0e-3)
    return Workload(f"cfg3_{n}_{prec}", "reservoir", prec, n, n, 1, dx, dx, prm, n_steps, P=P,
                    fields={"psi_p": psi, "n_p": np.zeros((1, n, n), dtype=rdt)})


def cfg4(n=16384, prec="c32", n_steps=2000, sigma_cells=50.0, tile=None):
    """Config 4: two-component spinor, TE-TM coupling, two Gaussian vortices of charge +1 / -1.

    tile=t (t divides n): the recipe is drawn on a t x t grid and repeated periodically to n x n -- a vortex lattice with
    the same value distribution, ready in seconds instead of a minute (used by bench.py's short other_workloads timings
    only; throughput does not depend on the field values)."""
    if tile is not None and tile != n:
        if n % tile != 0:
            raise ValueError("tile must divide n")
        w = cfg4(tile, prec, n_steps, sigma_cells)
        reps = n // tile
        w.fields = {k: np.tile(v, (1, reps, reps)) for k, v in w.fields.items()}
        w.name, w.nx, w.ny = f"cfg4_{n}_{prec}", n, n
        return w
    dx = 0.2
    cdt, rdt = _CDT[prec], _RDT[prec]
    rng = np.random.default_rng(3)
    sig = sigma_cells * dx
    x = ((np.arange(n) - n // 2) * dx)[None, :]
    fields = {}
    for name, sgn in (("psi_p", +1.0), ("psi_m", -1.0)):
        out = np.empty((1, n, n), dtype=cdt)
        for j0 in range(0, n, 256):
            j1 = min(n, j0 + 256)
            y = ((np.arange(j0, j1) - n // 2) * dx)[:, None]
            env = np.exp(-(x * x + y * y) / (2 * sig * sig)) / sig
            out[0, j0:j1] = ((x + sgn * 1j * y) * env).astype(cdt)
        out += _cnormal(rng, (1, n, n), 1e-3, cdt)
        fields[name] = out
    prm = dict(hbar=1.0, m=0.5, g=1e-3, g_x=2e-4, beta=0.1, gamma_c=0.05, dt=0.002)
    return Workload(f"cfg4_{n}_{prec}", "spinor", prec, n, n, 1, dx, dx, prm, n_steps, fields=fields)


def cfg5(n=256, batch=512, prec="c32", n_steps=20000, noise=True):
    """Config 5: Monte-Carlo (truncated Wigner) ensemble of `batch` n x n polariton grids with noise."""
    cdt, rdt = _CDT[prec], _RDT[prec]
    dx = 200.0 / n
    psi = np.empty((batch, n, n), dtype=cdt)
    for r in range(batch):
        psi[r] = _cnormal(np.random.default_rng([4, r]), (n, n), 1e-2, cdt)
    P = ring_pump(n, n, dx, dx, 100.0, 30.0, rdt)
    prm = dict(_POLARITON, dt=0.02, noise_scale=1.0)
    return Workload(f"cfg5_{batch}x{n}_{prec}", "reservoir", prec, n, n, batch, dx, dx, prm, n_steps, noise=noise,
                    seed=4, P=P, fields={"psi_p": psi, "n_p": np.zeros((batch, n, n), dtype=rdt)})


def example3(n=500, prec="c32", n_steps=1000):
    """spinor with reservoirs n+-, ring pump (the paper's Example 3 shape)."""
    cdt, rdt = _CDT[prec], _RDT[prec]
    dx = 0.2
    rng = np.random.default_rng(5)
    fields = {"psi_p": _cnormal(rng, (1, n, n), 1e-2, cdt), "psi_m": _cnormal(rng, (1, n, n), 1e-2, cdt),
              "n_p": np.zeros((1, n, n), dtype=rdt), "n_m": np.zeros((1, n, n), dtype=rdt)}
    P = ring_pump(n, n, dx, dx, 100.0, 0.15 * n * dx, rdt)
    prm = dict(_POLARITON, g_x=-1.2e-6, beta=2.5e-5, dt=0.01)
    return Workload(f"ex3_{n}_{prec}", "spinor_reservoir", prec, n, n, 1, dx, dx, prm, n_steps, P=P, fields=fields)
