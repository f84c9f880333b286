"""Shared helpers of the parity tests: run the same workload through libphx (CUDA) and the oracle (CPU)."""
import numpy as np


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    b = np.asarray(b, dtype=a.dtype)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


TOL = {"c32": 2e-5, "c64": 1e-12}   # BASELINE.json north_star: relative L2 after N steps

# Element-wise guard next to every relative-L2 bar: max |got - ref| <= ELEM_C * tol * max |ref|.  The L2 norm averages
# a localised error away (one wrong column of 4096 at relative size 1e-3 contributes 1.5e-5); rounding errors are spread
# evenly, so their largest element stays within a few standard deviations of the rms error (5.5 sigma over 1e7 cells)
# and rms |ref| <= max |ref|: a field inside the L2 bar is inside this one with ELEM_C = 8, a seam error is not.
ELEM_C = 8.0


def max_abs_ratio(a, b):
    """max |a - b| / max |b| (the element-wise error in units of the largest reference element)."""
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    b = np.asarray(b, dtype=a.dtype)
    return float(np.max(np.abs(a - b)) / max(float(np.max(np.abs(b))), 1e-300))


def check_close(got, ref, tol, what):
    """The two bars of every parity comparison: relative L2 <= tol and max |delta| <= ELEM_C tol max |ref|."""
    assert np.all(np.isfinite(got)), f"{what}: non-finite values on the GPU"
    err = rel_l2(got, ref)
    assert err <= tol, f"{what}: rel L2 {err:.3e} > {tol:.1e}"
    emax = max_abs_ratio(got, ref)
    assert emax <= ELEM_C * tol, f"{what}: max |delta| / max |ref| = {emax:.3e} > {ELEM_C * tol:.1e}"
    return err


def make_oracle(w, bc=(0, 0), E=None, extra_params=None):
    import oracle as orc
    prm = dict(w.params)
    if extra_params:
        prm.update(extra_params)
    o = orc.Oracle(w.nx, w.ny, w.dx, w.dy, orc.make_params(**prm), model=w.model, batch=w.batch,
                   prec32=(w.prec == "c32"), noise=w.noise, seed=w.seed, bc=bc,
                   V=None if w.V is None else w.V.astype(np.float64),
                   P=None if w.P is None else w.P.astype(np.float64),
                   E=None if E is None else E.astype(np.complex128))
    for name, arr in w.fields.items():
        o.set_field(name, arr)
    return o


def make_gpu(w, bc=(0, 0), E=None, extra_params=None, variant=0, tuning=None):
    from paper_2411_18341_b200 import binding as phx
    prm = dict(w.params)
    if extra_params:
        prm.update(extra_params)
    g = phx.Grid(w.nx, w.ny, w.dx, w.dy, model=w.model, prec=w.prec, batch=w.batch, noise=w.noise, bc=bc)
    g.set_params(phx.make_params(seed=w.seed, **prm))
    if w.V is not None or w.P is not None:
        g.set_potential_pump(w.V, w.P)
    if E is not None:
        g.set_drive(E)
    if variant:
        g.select_variant(variant)
    for k, v in (tuning or {}).items():
        g.set_tuning(k, v)
    for name, arr in w.fields.items():
        g.set_field(name, arr)
    return g


def compare(g, o, w, tol=None):
    """Element-wise comparison of every state field (relative L2 and largest element, check_close); returns dict
    field -> relative L2 error."""
    tol = TOL[w.prec] if tol is None else tol
    errs = {}
    for name in w.fields:
        errs[name] = check_close(g.read_field(name), getattr(o, name), tol, f"{w.name} {name}")
    return errs
