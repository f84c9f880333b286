"""Pins of the oracle's stochastic part (Eq. (22); BASELINE.json config 5)."""
import os

import numpy as np

import oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answer_vectors():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        w = [int(v, 16) for v in r]
        out = orc.philox4x32_10(w[0:4], w[4:6])
        assert [int(v) for v in out] == w[6:10]


def test_noise_words_are_keyed_by_seed_realisation_step_cell():
    nx, ny, B = 5, 4, 3
    step = (7 << 32) + 123456
    w = orc.noise_u32(nx, ny, B, seed=4, step=step)
    for r in (0, 2):
        for cell in (0, 7, nx * ny - 1):
            ref = orc.philox4x32_10([cell, step & 0xffffffff, step >> 32, 0], [4, r])
            assert np.array_equal(w[r].reshape(-1, 4)[cell], ref)
    assert len(np.unique(w)) == w.size                      # no repeated words across cells/realisations
    assert not np.array_equal(w, orc.noise_u32(nx, ny, B, seed=5, step=step))
    assert not np.array_equal(w, orc.noise_u32(nx, ny, B, seed=4, step=step + 1))


def test_uniform_map_is_exact_in_fp32_and_open_interval():
    for w0 in (0, 0x1ff, 0x200, 0xffffffff, 0x80000000, 0xfffffe00):
        u = ((w0 >> 9) + 0.5) / 8388608.0
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u
        xi1, xi2 = orc.normal_pair(w0, 0)                   # u2 = 2^-24: angle ~ 0
        assert abs(xi1 - np.sqrt(-2 * np.log(u)) * np.cos(2 * np.pi * 2.0 ** -24)) < 1e-15
        xi1, xi2 = orc.normal_pair(w0, 0x40000000)          # u2 = 0.25 + 2^-24: angle ~ pi/2
        assert abs(xi2 - np.sqrt(-2 * np.log(u)) * np.sin(2 * np.pi * (0.25 + 2.0 ** -24))) < 1e-15


def test_noise_moments_match_eq22():
    # psi = 0, no reservoir dynamics: after one step psi = sigma (xi1 + i xi2) with
    # sigma^2 = nu dt gamma_c / (4 dx dy) per real component, <dW dW*> = 2 sigma^2, <dW dW> = 0.
    nx = ny = 64
    B, dx, dy, dt, gam, nu = 64, 0.5, 0.8, 0.02, 0.15, 1.7
    o = orc.Oracle(nx, ny, dx, dy, orc.make_params(gamma_c=gam, dt=dt, noise_scale=nu), batch=B, noise=True, seed=4)
    o.step_rk4(1)
    z = o.psi_p.ravel()
    sig2 = nu * dt * gam / (4 * dx * dy)
    n = z.size
    assert abs(z.real.mean()) < 5 * np.sqrt(sig2 / n) and abs(z.imag.mean()) < 5 * np.sqrt(sig2 / n)
    assert abs(z.real.var() / sig2 - 1) < 5 * np.sqrt(2 / n) and abs(z.imag.var() / sig2 - 1) < 5 * np.sqrt(2 / n)
    assert abs(np.mean(z * z)) < 5 * 2 * sig2 / np.sqrt(n)                       # <dW dW> = 0
    assert abs(np.mean(np.abs(z) ** 2) / (2 * sig2) - 1) < 5 / np.sqrt(n)        # <dW dW*> = 2 sigma^2
    kurt = np.mean(z.real ** 4) / sig2 ** 2
    assert abs(kurt - 3) < 5 * np.sqrt(96 / n)
    # spatial delta correlation: neighbouring cells uncorrelated
    f = o.psi_p
    assert abs(np.mean(f[:, :, 1:] * np.conj(f[:, :, :-1]))) < 5 * 2 * sig2 / np.sqrt(n)


def test_noise_uses_reservoir_before_the_step_and_stream_of_each_realisation():
    nx, ny, B = 8, 6, 4
    rng = np.random.default_rng(20)
    P = rng.uniform(0, 50, (ny, nx))
    n0 = rng.uniform(0, 40, (B, ny, nx))
    dx, dt = 0.78125, 0.02
    prm = orc.make_params(hbar=6.582e-4, m=5.7e-4, g=6e-6, g_r=12e-6, R=0.01, gamma_c=0.15, gamma_r=0.225, dt=dt)
    step0 = 11
    det = orc.Oracle(nx, ny, dx, dx, prm, model="reservoir", batch=B, P=P)
    sto = orc.Oracle(nx, ny, dx, dx, prm, model="reservoir", batch=B, P=P, noise=True, seed=4)
    for o in (det, sto):
        o.set_field("n_p", n0)
        o.step = step0
        o.step_rk4(1)
    words = orc.noise_u32(nx, ny, B, 4, step0)
    xi = np.array([orc.normal_pair(int(w[0]), int(w[1])) for w in words.reshape(-1, 4)]).reshape(B, ny, nx, 2)
    sigma = np.sqrt(dt / (4 * dx * dx) * (0.15 + 0.01 * n0))
    expect = det.psi_p + sigma * (xi[..., 0] + 1j * xi[..., 1])
    assert np.allclose(sto.psi_p, expect, rtol=0, atol=1e-15)
    assert np.array_equal(sto.n_p, det.n_p)


def test_noise_scale_zero_is_deterministic_and_spinor_uses_words_2_3():
    nx, ny = 6, 6
    rng = np.random.default_rng(21)
    a = 0.3 * (rng.standard_normal((1, ny, nx)) + 1j * rng.standard_normal((1, ny, nx)))
    prm0 = orc.make_params(g=0.5, gamma_c=0.2, dt=0.01, noise_scale=0.0)
    o0 = orc.Oracle(nx, ny, 0.5, 0.5, prm0, noise=True, seed=9)
    o1 = orc.Oracle(nx, ny, 0.5, 0.5, prm0)
    for o in (o0, o1):
        o.set_field("psi_p", a)
        o.step_rk4(5)
    assert np.array_equal(o0.psi_p, o1.psi_p)
    prm = orc.make_params(gamma_c=0.2, dt=0.01)
    sp = orc.Oracle(nx, ny, 0.5, 0.5, prm, model="spinor", noise=True, seed=9)
    sp.step_rk4(1)
    w = orc.noise_u32(nx, ny, 1, 9, 0).reshape(-1, 4)
    sig = np.sqrt(0.01 * 0.2 / (4 * 0.25))
    for name, k in (("psi_p", 0), ("psi_m", 2)):
        xi = np.array([orc.normal_pair(int(v[k]), int(v[k + 1])) for v in w])
        assert np.allclose(getattr(sp, name).ravel(), sig * (xi[:, 0] + 1j * xi[:, 1]), rtol=0, atol=1e-16)


def test_ensemble_mean_density():
    rng = np.random.default_rng(22)
    B, ny, nx = 5, 4, 3
    o = orc.Oracle(nx, ny, 1.0, 1.0, orc.make_params(dt=0.1), batch=B)
    a = rng.standard_normal((B, ny, nx)) + 1j * rng.standard_normal((B, ny, nx))
    o.set_field("psi_p", a)
    assert np.allclose(o.ensemble_mean_density(), (np.abs(a) ** 2).mean(axis=0), rtol=1e-15)


def test_philox_matches_curand_header_on_random_inputs(tmp_path):
    """Independent implementation: cuRAND's curand_Philox4x32_10 compiled for the host."""
    import ctypes as C
    import subprocess
    import pytest
    cuda_inc = "/usr/local/cuda/include"
    if not os.path.exists(os.path.join(cuda_inc, "curand_philox4x32_x.h")):
        pytest.skip("cuRAND headers not present")
    so = str(tmp_path / "libcph.so")
    src = os.path.join(os.path.dirname(__file__), "curand_philox_host.cpp")
    subprocess.run(["g++", "-O1", "-shared", "-fPIC", "-I" + cuda_inc, "-o", so, src], check=True)
    lib = C.CDLL(so)
    rng = np.random.default_rng(23)
    n = 20000
    ctr = rng.integers(0, 2 ** 32, (n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, (n, 2), dtype=np.uint64).astype(np.uint32)
    ref = np.zeros((n, 4), np.uint32)
    lib.curand_philox_host(ctr.ctypes.data_as(C.c_void_p), key.ctypes.data_as(C.c_void_p),
                           ref.ctypes.data_as(C.c_void_p), C.c_int64(n))
    got = np.array([orc.philox4x32_10(ctr[i], key[i]) for i in range(n)])
    assert np.array_equal(got, ref)


def test_first_realisation_offsets_the_philox_key():
    # element r of a batch == a batch of one with first_realisation = r (used to step single realisations of cfg5)
    prm = orc.make_params(g=0.5, gamma_c=0.1, R=0.01, gamma_r=0.2, dt=0.02)
    rng = np.random.default_rng(40)
    a = rng.standard_normal((3, 6, 5)) + 1j * rng.standard_normal((3, 6, 5))
    ob = orc.Oracle(5, 6, 0.5, 0.5, prm, model="reservoir", batch=3, noise=True, seed=9, P=np.ones((6, 5)))
    ob.set_field("psi_p", a)
    ob.step_rk4(4)
    for r in range(3):
        o1 = orc.Oracle(5, 6, 0.5, 0.5, prm, model="reservoir", batch=1, noise=True, seed=9, P=np.ones((6, 5)),
                        first_realisation=r)
        o1.set_field("psi_p", a[r:r + 1])
        o1.step_rk4(4)
        assert np.array_equal(o1.psi_p[0], ob.psi_p[r]) and np.array_equal(o1.n_p[0], ob.n_p[r])
