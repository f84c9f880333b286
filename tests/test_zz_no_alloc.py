"""phx_step_rk4_static (include/phx.h): RK4 steps without a handle, a workspace or any allocation -- the stage buffers live in a
file-scope device array inside libphx.so (paper_2411_18341_b200/csrc/phx_static.cu).  Checked against the existing path
(a phx_grid handle stepping with the same per-stage kernels, variant STAGE) within the tolerances of the other parity tests,
on two calls in a row, with stale contents of the shared array in between, and for the size limit.
Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`."""
import numpy as np
import pytest

from paper_2411_18341_b200 import workloads as wl
from helpers import TOL, check_close, make_gpu

pytestmark = pytest.mark.gpu
STAGE = 1


def _device_inputs(w):
    import torch
    psi = torch.from_numpy(np.ascontiguousarray(w.fields["psi_p"][0])).cuda()
    V = None if w.V is None else torch.from_numpy(np.ascontiguousarray(w.V)).cuda()
    return psi, V


def _params(w):
    from paper_2411_18341_b200 import binding as phx
    return phx.make_params(seed=w.seed, **w.params)


def _existing_path(w, n_steps, bc=(0, 0)):
    g = make_gpu(w, variant=STAGE, bc=bc)
    g.step_rk4(n_steps)
    out = g.read_field("psi_p")[0]
    g.destroy()
    return out


@pytest.mark.parametrize("prec,nx,ny,bc", [("c32", 256, 192, (0, 0)), ("c64", 200, 75, (0, 0)), ("c32", 131, 67, (1, 0)),
                                            ("c64", 64, 64, (1, 1))])
def test_static_entry_point_matches_the_handle_path_on_two_calls_in_a_row(prec, nx, ny, bc):
    import torch
    from paper_2411_18341_b200 import binding as phx
    w = wl.cfg2(n=nx, ny=ny, prec=prec)
    ref10, ref20 = _existing_path(w, 10, bc), _existing_path(w, 20, bc)
    psi0, V = _device_inputs(w)
    prm = _params(w)
    out = torch.empty_like(psi0)
    # call 1: out <- 10 steps of psi0; call 2 (in place, directly after it on the same stream): 10 more
    phx.step_rk4_static(psi0, out, w.dx, w.dy, prm, V=V, n_steps=10, bc=bc)
    torch.cuda.synchronize()
    check_close(out.cpu().numpy(), ref10, TOL[prec], f"static {w.name} bc {bc}, call 1")
    phx.step_rk4_static(out, out, w.dx, w.dy, prm, V=V, n_steps=10, bc=bc)
    torch.cuda.synchronize()
    got20 = out.cpu().numpy()
    check_close(got20, ref20, TOL[prec], f"static {w.name} bc {bc}, call 2")
    assert np.array_equal(psi0.cpu().numpy(), w.fields["psi_p"][0])           # the input array is the caller's: untouched
    # the shared array keeps the last call's contents: a call on another grid in between must not change the next result
    w2 = wl.cfg2(n=96, ny=40, prec=prec)
    p2, V2 = _device_inputs(w2)
    o2 = torch.empty_like(p2)
    phx.step_rk4_static(p2, o2, w2.dx, w2.dy, _params(w2), V=V2, n_steps=3)
    check_close(o2.cpu().numpy(), _existing_path(w2, 3), TOL[prec], "static, other grid in between")
    out2 = torch.empty_like(psi0)
    phx.step_rk4_static(psi0, out2, w.dx, w.dy, prm, V=V, n_steps=20, bc=bc)
    torch.cuda.synchronize()
    assert np.array_equal(out2.cpu().numpy(), got20)                            # one call of 20 steps = two of 10, bit for bit


def test_static_entry_point_allocates_no_device_memory_and_enqueues_on_the_callers_stream():
    import torch
    from paper_2411_18341_b200 import binding as phx
    w = wl.cfg2(n=128, ny=128, prec="c32")
    psi0, V = _device_inputs(w)
    prm = _params(w)
    out = torch.empty_like(psi0)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    phx.step_rk4_static(psi0, out, w.dx, w.dy, prm, V=V, n_steps=2, stream=stream)    # (first use loads the kernels' module)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        phx.step_rk4_static(psi0, out, w.dx, w.dy, prm, V=V, n_steps=5, stream=stream)
    stream.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "the device's free memory changed across phx_step_rk4_static calls"
    check_close(out.cpu().numpy(), _existing_path(w, 5), TOL["c32"], "static on a side stream")


def test_static_entry_point_rejects_grids_beyond_the_scratch_array_and_bad_arguments():
    import torch
    from paper_2411_18341_b200 import binding as phx
    prm = phx.make_params(hbar=1.0, m=0.5, g=2e-3, gamma_c=0.1, dt=0.004)
    for dtype, n in ((torch.complex64, 600), (torch.complex128, 420), (torch.complex64, 4096)):
        psi = torch.zeros((n, n), dtype=dtype, device="cuda")
        out = torch.full_like(psi, 7.0)
        with pytest.raises(phx.PhxError) as e:
            phx.step_rk4_static(psi, out, 0.2, 0.2, prm, n_steps=1)
        assert e.value.status == phx.PHX_ERR_WORKSPACE and "static array holds" in str(e.value)
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())                                        # nothing was enqueued
        del psi, out
    # the largest square grids that fit: 590^2 complex fp32, 417^2 complex fp64
    for dtype, n in ((torch.complex64, 590), (torch.complex128, 417)):
        psi = torch.zeros((n, n), dtype=dtype, device="cuda")
        phx.step_rk4_static(psi, psi, 0.2, 0.2, prm, n_steps=1)
        torch.cuda.synchronize()
        assert bool((psi == 0).all())
    small = torch.zeros((8, 8), dtype=torch.complex64, device="cuda")
    with pytest.raises(phx.PhxError) as e:
        phx.step_rk4_static(small, small, 0.2, 0.2, phx.make_params(hbar=1.0, m=0.5, dt=0.0), n_steps=1)      # dt must be > 0
    assert e.value.status == phx.PHX_ERR_INVALID_ARG
    with pytest.raises(phx.PhxError) as e:
        phx.step_rk4_static(small[:2, :2].contiguous(), small, 0.2, 0.2, prm, n_steps=1)                      # nx, ny >= 3
    assert e.value.status == phx.PHX_ERR_INVALID_ARG
