"""Builds paper_2411_18341_b200/libphx.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2411_18341_b200.build [--force] [--verbose]
"""
import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libphx.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
         "-Xcompiler", "-fPIC", "-I", INCLUDE, "-I", CSRC] + os.environ.get("PHX_NVCC_EXTRA", "").split()


def _units():
    """(object name, source, extra defines)"""
    u = [("phx_api.o", "phx_api.cu", []), ("phx_aux.o", "phx_aux.cu", []), ("phx_resident.o", "phx_resident.cu", []),
         ("phx_adaptive.o", "phx_adaptive.cu", []), ("phx_static.o", "phx_static.cu", [])]
    for prec in (32, 64):
        for model in range(4):
            u.append((f"phx_stage_{prec}_{model}.o", "phx_stage_inst.cu",
                      [f"-DPHX_INST_PREC={prec}", f"-DPHX_INST_MODEL={model}"]))
            u.append((f"phx_step_{prec}_{model}.o", "phx_step_inst.cu",
                      [f"-DPHX_INST_PREC={prec}", f"-DPHX_INST_MODEL={model}"]))
            if model < 2:
                u.append((f"phx_stepx_{prec}_{model}.o", "phx_stepx_inst.cu",
                          [f"-DPHX_INST_PREC={prec}", f"-DPHX_INST_MODEL={model}"]))
    return u


def _sources_digest():
    h = hashlib.sha256()
    for root in (CSRC, INCLUDE):
        for name in sorted(os.listdir(root)):
            with open(os.path.join(root, name), "rb") as f:
                h.update(name.encode())
                h.update(f.read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "digest.txt")
    digest = _sources_digest()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == digest:
        return LIB
    units = _units()

    def compile_one(u):
        obj, src, defs = u
        cmd = [NVCC] + FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o",
                                                                                 os.path.join(OBJ, obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return obj, r.returncode, r.stdout + r.stderr

    with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        results = list(ex.map(compile_one, units))
    for obj, rc, out in results:
        if verbose or rc != 0:
            sys.stderr.write(f"--- {obj}\n{out}\n")
        if rc != 0:
            raise RuntimeError(f"nvcc failed for {obj}")
    cmd = [NVCC, "-shared", "-o", LIB] + [os.path.join(OBJ, u[0]) for u in units] + ["-lcudart"]
    subprocess.run(cmd, check=True)
    with open(stamp, "w") as f:
        f.write(digest)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
