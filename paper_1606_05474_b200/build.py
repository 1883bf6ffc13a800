"""Builds libhelios_b200.so (the C-ABI library of include/helios.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The library is rebuilt when the content of any source under csrc/ or of
include/helios.h differs from what the existing .so was built from.

  python -m paper_1606_05474_b200.build [--force] [-v] [--dev] [--checked]

The ray kernel (csrc/helios_flux.cu) is compiled once per unit = (variant, arithmetic, lanes per ray): 18
translation units, in parallel.  --dev (developer builds only; never used by build() as the driver or the
binding call it): instantiates just the shapes of the BASELINE configs and of the parity tests, which compiles in
a fraction of the time; such a library is marked and is replaced by a full one the next time
__graft_entry__.build() or `python -m paper_1606_05474_b200.build` runs without --dev.  --checked (implies --dev): the ray
kernel's own memory checker (HX_CHECKED in csrc/helios_flux.cu: NaN-poisoned shared memory, guard words, index
checks), for `python -m paper_1606_05474_b200.selfcheck` where compute-sanitizer is not available.
"""
from __future__ import annotations

import glob
import hashlib
import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libhelios_b200.so")
HASH = LIB + ".srchash"
PLAIN_SOURCES = ["helios_api.cu", "helios_aux.cu", "helios_flux_dispatch.cu"]
FLUX_SOURCE = "helios_flux.cu"
# (variant, fp32, lanes per ray) -> one object file each
FLUX_UNITS = [(alt, f32, lpr) for alt in (0, 1, 2) for f32 in (0, 1) for lpr in (8, 16, 32)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")
    return exe


def _source_hash() -> str:
    """Content hash of everything the library is built from (sources, header, flags): file times do
    not survive copying the tree to another machine, contents do."""
    h = hashlib.sha256()
    deps = sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + glob.glob(os.path.join(CSRC, "*.h")) + [os.path.join(ROOT, "include", "helios.h")])
    for d in deps:
        h.update(os.path.basename(d).encode())
        h.update(open(d, "rb").read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def _recorded():
    """(source hash, 'full' | 'dev') the existing library was built from, or (None, None)."""
    if not os.path.exists(LIB) or not os.path.exists(HASH):
        return None, None
    parts = open(HASH).read().split()
    return (parts[0], parts[1] if len(parts) > 1 else "full") if parts else (None, None)


def _stale(accept_dev: bool) -> bool:
    h, kind = _recorded()
    return h != _source_hash() or (kind == "dev" and not accept_dev)


def build(force: bool = False, verbose: bool = False, dev: bool = False, accept_dev: bool = False,
          checked: bool = False) -> str:
    """Full build unless dev=True.  accept_dev: an up-to-date developer build counts as current (the binding
    passes this so that a developer's test run does not trigger the long build; __graft_entry__.build() does not)."""
    if not force and not _stale(accept_dev or dev):
        return LIB
    jobs = []
    dev = dev or checked
    extra = os.environ.get("HELIOS_DEV_DEFS", "").split() if dev else []     # experiments of developer builds only
    if checked:
        extra.append("-DHX_CHECKED")
    for src in PLAIN_SOURCES:
        jobs.append((os.path.join(CSRC, src), os.path.join(CSRC, src.replace(".cu", ".o")), extra))
    for alt, f32, lpr in FLUX_UNITS:
        defs = [f"-DHX_FLUX_ALT={alt}", f"-DHX_FLUX_F32={f32}", f"-DHX_FLUX_LPR={lpr}"] + (["-DHX_DEV_SHAPES"] + extra if dev else [])
        jobs.append((os.path.join(CSRC, FLUX_SOURCE), os.path.join(CSRC, f"helios_flux_v{alt}_f{f32}_l{lpr}.o"), defs))
    for stale_obj in glob.glob(os.path.join(CSRC, "*.o")):
        os.remove(stale_obj)
    workers = max(1, os.cpu_count() or 1)
    running, objs, todo = [], [o for _, o, _ in jobs], list(jobs)

    def reap(block):
        for item in list(running):
            cmd, pr = item
            if block or pr.poll() is not None:
                out, _ = pr.communicate()
                running.remove(item)
                if verbose and out:
                    print(out)
                if pr.returncode != 0:
                    for _, other in running:
                        other.kill()
                    raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + (out or ""))
                if block:
                    return

    while todo or running:
        while todo and len(running) < workers:
            src, obj, defs = todo.pop(0)
            cmd = [nvcc(), *NVCC_FLAGS, *defs, "-c", src, "-o", obj]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            running.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        reap(block=True)
    link = [nvcc(), "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a",
            "-Xcompiler", "-fPIC", "-lcudart"]
    subprocess.check_call(link)
    with open(HASH, "w") as f:
        f.write(_source_hash() + (" dev" if dev else " full"))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or "--checked" in sys.argv, verbose="-v" in sys.argv, dev="--dev" in sys.argv,
                checked="--checked" in sys.argv))
