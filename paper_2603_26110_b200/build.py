"""In-tree build of libtq.so (nvcc, sm_100a only).  `python -m paper_2603_26110_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtq.so")
SOURCES = ["tq_api.cu", "tq_layout.cu", "tq_quantize.cu", "tq_quantize_tc.cu", "tq_decode.cu", "tq_prep.cu", "tq_calibrate_host.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC",
              "--expt-relaxed-constexpr"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "tq.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, test_hooks: bool = True) -> str:
    """test_hooks = True (what the tests, bench.py and __graft_entry__ build): libtq.so with -DTQ_TEST_HOOKS, i.e. with
    tq_profile_decode_main_only, tq_debug_set_decode_nsplit, tq_debug_set_quantize_impl and the fp32 cross-check kernel.
    test_hooks = False (`python -m paper_2603_26110_b200.build --product`): build/libtq_product.so without them — no
    measurement or test switch, no process-wide mutable state on the product path."""
    lib = LIB if test_hooks else os.path.join(HERE, "build", "libtq_product.so")
    if test_hooks and not force and not _stale():
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = ["-DTQ_TEST_HOOKS"] if test_hooks else []
    objs = []
    procs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src + (".o" if test_hooks else ".product.o"))
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(out)
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", lib, *objs, "-lcudart"], check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, test_hooks="--product" not in sys.argv))
