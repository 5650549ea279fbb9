"""Build step for the CUDA library (nvcc, sm_100a only).  `python -m paper_2506_21804_b200.build [--force] [-v]`.

csrc/lbm_api.cu (host side of the C ABI, set-up kernels) + csrc/lbm_static.cu (lbm_totals_static: static device scratch, nothing
allocated) + csrc/lbm_inst.cu compiled once per (lattice, dtype, part): eighteen
object files, built in parallel, linked into liblbm_b200.so next to this file."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
OBJ = os.path.join(PKG, "build")
LIB = os.path.join(PKG, "liblbm_b200.so")
HEADERS = ["lbm_kernels.cuh", "lbm_launch.cuh", "lbm_ctx.h", os.path.join("..", "..", "include", "lbm.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC"]
# (object name, source, defines)
UNITS = [("lbm_api", "lbm_api.cu", []), ("lbm_static", "lbm_static.cu", [])]
for _q in (19, 27):
    for _t in ("float", "double"):
        for _part in (0, 1, 2, 3):
            UNITS.append(("lbm_inst_q%d_%s_p%d" % (_q, _t, _part), "lbm_inst.cu",
                          ["-DLBM_INST_Q=%d" % _q, "-DLBM_INST_T=%s" % _t, "-DLBM_INST_PART=%d" % _part]))


def _deps(src):
    return [os.path.join(CSRC, src)] + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(unit, verbose):
    name, src, defs = unit
    obj = os.path.join(OBJ, name + ".o")
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return name, res


def build(force=False, verbose=False, jobs=None):
    """Compile csrc/*.cu into liblbm_b200.so next to this file.  Returns the library path."""
    os.makedirs(OBJ, exist_ok=True)
    todo = [u for u in UNITS if force or _stale(os.path.join(OBJ, u[0] + ".o"), _deps(u[1]))]
    if todo:
        jobs = jobs or int(os.environ.get("LBM_BUILD_JOBS", str(os.cpu_count() or 4)))
        with ThreadPoolExecutor(max_workers=max(1, jobs)) as ex:
            results = list(ex.map(lambda u: _compile(u, verbose), todo))
        failed = [(n, r) for n, r in results if r.returncode != 0]
        for n, r in results:
            if verbose or r.returncode != 0:
                sys.stderr.write("==== %s\n%s%s" % (n, r.stdout, r.stderr))
        if failed:
            for n, _ in failed:
                try:
                    os.remove(os.path.join(OBJ, n + ".o"))
                except OSError:
                    pass
            raise RuntimeError("nvcc failed building %s" % ", ".join(n for n, _ in failed))
    objs = [os.path.join(OBJ, u[0] + ".o") for u in UNITS]
    if todo or _stale(LIB, objs):
        nvcc = os.environ.get("NVCC", "nvcc")
        tmp = LIB + ".tmp.%d" % os.getpid()
        res = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs,
                             capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("link failed for %s" % LIB)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
