"""Shared helpers of the parity tests: run the same workload through libphx (CUDA) and the oracle (CPU)."""
import numpy as np


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) else np.float64)
    b = np.asarray(b, dtype=a.dtype)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


TOL = {"c32": 2e-5, "c64": 1e-12}   # BASELINE.json north_star: relative L2 after N steps


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
    """Element-wise comparison of every state field; returns dict field -> relative L2 error."""
    tol = TOL[w.prec] if tol is None else tol
    errs = {}
    for name in w.fields:
        got = g.read_field(name)
        ref = getattr(o, name)
        errs[name] = rel_l2(got, ref)
        assert np.all(np.isfinite(got)), f"{name}: non-finite values on the GPU"
        assert errs[name] <= tol, f"{w.name} {name}: rel L2 {errs[name]:.3e} > {tol:.1e}"
    return errs
