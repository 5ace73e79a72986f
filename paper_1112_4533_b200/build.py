"""Build libsugauge.so (sm_100a) in-tree:  python -m paper_1112_4533_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU. One object per (translation unit, Nc) so the compile parallelises;
objects are cached under csrc/build/ keyed by the sources' mtimes.
"""
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# SUG_BUILD_VARIANT=<name> with SUG_NVCC_EXTRA="-D..." builds libsugauge_<name>.so next to the product library
# (tuning / ablation builds, e.g. -DSUG_LINK_TILE=1); the product build uses neither.
VARIANT = os.environ.get("SUG_BUILD_VARIANT", "")
EXTRA = os.environ.get("SUG_NVCC_EXTRA", "").split() if VARIANT else []
OBJ = os.path.join(CSRC, "build" + ("_" + VARIANT if VARIANT else ""))
LIB = os.path.join(HERE, "libsugauge" + ("_" + VARIANT if VARIANT else "") + ".so")
NCS = list(range(2, 9))

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
]
HEADERS = ["su_device.cuh", "su_internal.h", "update_kernel.cuh", "update_rows_kernel.cuh", "fused_schedule.h", os.path.join("..", "..", "include", "su_gauge.h"),
           os.path.join("..", "..", "include", "su_gauge_test.h")]


def _units():
    units = [("su_api.cu", None), ("fused_schedule.cu", None), ("big_kernels.cu", None), ("static_scratch.cu", None)]
    for nc in NCS:
        units.append(("update_kernels.cu", nc))
        units.append(("aux_kernels.cu", nc))
    return units


def _newest_header():
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _compile(unit, force, verbose):
    src, nc = unit
    obj = os.path.join(OBJ, src.replace(".cu", "") + (f"_nc{nc}" if nc else "") + ".o")
    srcp = os.path.join(CSRC, src)
    if (not force and os.path.exists(obj)
            and os.path.getmtime(obj) >= max(os.path.getmtime(srcp), _newest_header())):
        return obj, ""
    cmd = ["nvcc", *NVCC_FLAGS, *EXTRA, "-c", srcp, "-o", obj]
    if nc:
        cmd.append(f"-DSUG_NC={nc}")
    if verbose:
        cmd += ["-Xptxas", "-v"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {src} (Nc={nc}):\n{r.stdout}\n{r.stderr}")
    return obj, r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    units = _units()
    with cf.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        results = list(ex.map(lambda u: _compile(u, force, verbose), units))
    objs = [o for o, _ in results]
    if verbose:
        for _, log in results:
            sys.stderr.write(log)
    if force or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB, *objs]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
