"""Build libdisc.so (the C-ABI library of include/disc.h) with nvcc for sm_100a, in-tree.

The kernel templates are instantiated in several translation units (ranges of the patch radius R and of
the Gaussian radius K) that compile in parallel; the objects are linked into
`paper_1204_6295_b200/libdisc.so`.  Cross-compiles without a GPU.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdisc.so")

# no --use_fast_math: IEEE division and sqrt are kept
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]

R_RANGES = [(0, 3), (4, 6), (7, 9), (10, 12)]
K_RANGES = [(1, 3), (4, 6), (7, 9), (10, 12)]

def _units():
    units = [("disc_api", "disc_api.cu", [])]
    for i, (lo, hi) in enumerate(R_RANGES):
        units.append((f"moments_tu{i}", "moments_tu.cu", [f"-DDISC_TU={i}", f"-DDISC_R_LO={lo}", f"-DDISC_R_HI={hi}"]))
    for i, (lo, hi) in enumerate(K_RANGES):
        units.append((f"field_tu{i}", "field_tu.cu", [f"-DDISC_TU={i}", f"-DDISC_K_LO={lo}", f"-DDISC_K_HI={hi}"]))
    return units


def _source_hash() -> str:
    h = hashlib.sha256()
    for root in (CSRC, os.path.join(HERE, "..", "include")):
        for name in sorted(os.listdir(root)):
            with open(os.path.join(root, name), "rb") as f:
                h.update(name.encode())
                h.update(f.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    h.update(repr((R_RANGES, K_RANGES)).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False, ptxas_log: str | None = None) -> str:
    stamp = os.path.join(OBJ, "stamp")
    digest = _source_hash()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == digest:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = ["-Xptxas", "-v"] if ptxas_log else []

    def compile_one(unit):
        name, src, defs = unit
        obj = os.path.join(OBJ, name + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *extra, *defs, "-c", os.path.join(CSRC, src), "-o", obj]
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}:\n{p.stderr}")
        return obj, p.stderr

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, _units()))
    if ptxas_log:
        with open(ptxas_log, "w") as f:
            for _, err in results:
                f.write(err)
    objs = [o for o, _ in results]
    p = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs],
                       capture_output=True, text=True)
    if p.returncode != 0:
        raise RuntimeError(f"link failed:\n{p.stderr}")
    with open(stamp, "w") as f:
        f.write(digest)
    if verbose:
        print(f"built {LIB}", file=sys.stderr)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True,
          ptxas_log=next((a.split("=", 1)[1] for a in sys.argv if a.startswith("--ptxas-log=")), None))
