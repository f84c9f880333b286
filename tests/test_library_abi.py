"""CPU-side checks of the boundary: libphx.so builds, loads and exports every symbol include/phx.h declares.
No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2411_18341_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "phx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(phx_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_baseline_entry_points():
    syms = declared_symbols()
    for name in ("phx_create_grid", "phx_set_params", "phx_set_potential_pump", "phx_step_rk4", "phx_read_field",
                 "phx_set_field"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    lib = C.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(lib, name), f"libphx.so does not export {name}"


def test_binding_lists_the_same_names(libpath):
    from paper_2411_18341_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    binding.lib()


def test_struct_layouts_match_header(libpath, tmp_path):
    """Compile a tiny C program against include/phx.h and compare sizeof/offsetof with the ctypes mirrors."""
    import subprocess
    from paper_2411_18341_b200 import binding
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "phx.h"\nint main(void){\n'
                   'printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(phx_grid_desc), offsetof(phx_grid_desc, dx), '
                   'offsetof(phx_grid_desc, prec), offsetof(phx_grid_desc, workspace), offsetof(phx_grid_desc, stream), '
                   'sizeof(phx_params), offsetof(phx_params, seed), offsetof(phx_grid_desc, integrator), sizeof(phx_adaptive), '
                   'sizeof(phx_adaptive_state));\nreturn 0;}\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)], check=True)
    got = [int(v) for v in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    d, p = binding.phx_grid_desc, binding.phx_params
    assert got == [C.sizeof(d), d.dx.offset, d.prec.offset, d.workspace.offset, d.stream.offset, C.sizeof(p),
                   p.seed.offset, d.integrator.offset, C.sizeof(binding.phx_adaptive), C.sizeof(binding.phx_adaptive_state)]
    # the adaptive integrator's K buffers are reserved only when asked for
    rk = binding.phx_grid_desc(64, 64, 1, 0.5, 0.5, 0, 0, 0, 0, 0, 0, None, 0, None)
    dp = binding.phx_grid_desc(64, 64, 1, 0.5, 0.5, 0, 0, 0, 0, 0, 1, None, 0, None)
    lib = binding.lib()
    assert lib.phx_workspace_bytes(C.byref(dp)) >= lib.phx_workspace_bytes(C.byref(rk)) + 7 * 64 * 64 * 8


def test_invalid_descriptor_and_no_device_fail_loudly(libpath):
    from paper_2411_18341_b200 import binding
    lib = binding.lib()
    bad = binding.phx_grid_desc(2, 64, 1, 0.5, 0.5, 0, 0, 0, 0, 0, 0, None, 0, None)
    assert lib.phx_workspace_bytes(C.byref(bad)) == 0
    ok = binding.phx_grid_desc(64, 64, 1, 0.5, 0.5, 0, 0, 0, 0, 0, 0, None, 0, None)
    n = lib.phx_workspace_bytes(C.byref(ok))
    assert n >= 64 * 64 * 8 * 4
    # plane sizes up to 2^32 - 1 cells are admitted (the noise counter holds the cell index in 32 bits); the sizes are
    # computed in size_t: a 50 000^2 complex fp32 scalar grid needs 4 complex planes + V, P, E
    big = binding.phx_grid_desc(50000, 50000, 1, 0.5, 0.5, 0, 0, 1, 0, 0, 0, None, 0, None)
    nb = lib.phx_workspace_bytes(C.byref(big))
    assert nb >= 4 * 50000 * 50000 * 8 and nb < 8 * 50000 * 50000 * 8
    too_big = binding.phx_grid_desc(70000, 70000, 1, 0.5, 0.5, 0, 0, 0, 0, 0, 0, None, 0, None)
    assert lib.phx_workspace_bytes(C.byref(too_big)) == 0
    import torch
    if not torch.cuda.is_available():
        h = C.c_void_p()
        st = lib.phx_create_grid(C.byref(h), C.byref(ok))
        assert st != 0 and not h.value                      # no CPU fallback
        with pytest.raises(RuntimeError):
            binding.Grid(64, 64, 0.5, 0.5)
