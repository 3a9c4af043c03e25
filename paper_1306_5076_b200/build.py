"""Build libbcf.so (the C-ABI CUDA library, include/bcf.h) in-tree with nvcc for sm_100a.

Usage: python -m paper_1306_5076_b200.build [--force] [-v]      (also called by __graft_entry__.build()).
nvcc cross-compiles without a GPU.  The library is several translation units (csrc/bcf_api.cu = the C ABI and
the driver, csrc/bcf_tu_*.cu = one kernel family each) compiled in parallel into build/*.o and linked into
libbcf.so; a unit is recompiled when its source, a header under csrc/ or include/bcf.h is newer than its
object.  Objects and the .so are git-ignored; the .so travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
OUT = os.path.join(HERE, "libbcf.so")
SOURCES = ["bcf_api.cu", "bcf_tu_tile.cu", "bcf_tu_long.cu", "bcf_tu_merge.cu", "bcf_tu_pipe.cu", "bcf_tu_merge4.cu",
           "bcf_tu_buckets.cu", "bcf_tu_isolate.cu", "bcf_tu_static.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC",
]


def _headers_mtime():
    newest = os.path.getmtime(os.path.join(HERE, "..", "include", "bcf.h"))
    for f in os.listdir(CSRC):
        if f.endswith((".cuh", ".h")):
            newest = max(newest, os.path.getmtime(os.path.join(CSRC, f)))
    return newest


def _compile(nvcc, src, obj, verbose, extra):
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    r = subprocess.run(cmd, cwd=HERE, capture_output=True, text=True)
    return src, r.returncode, r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False, extra_flags=(), log=None) -> str:
    """Compile what is out of date and link.  `extra_flags` (e.g. -D...) are for A/B experiments only.  The flag set
    of the objects under build/ is recorded in build/flags.stamp; whenever it differs from this call's flags (in
    either direction) every unit is recompiled.  `log`: file that receives the compiler output (ptxas -v lines with
    verbose)."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    hdr = _headers_mtime()
    # The objects in build/ belong to ONE flag set.  Its record sits beside them; a build with other flags (an A/B
    # experiment with -D..., or the plain build that follows one) recompiles every unit instead of linking stale
    # objects of the other kernel shape into libbcf.so.
    flags_now = " ".join(NVCC_FLAGS + list(extra_flags))
    stamp = os.path.join(OBJ, "flags.stamp")
    try:
        with open(stamp) as f:
            flags_then = f.read()
    except OSError:
        flags_then = None
    if flags_then != flags_now:
        force = True
        for stale in [OUT] + [os.path.join(OBJ, f) for f in os.listdir(OBJ) if f.endswith(".o")]:
            if os.path.exists(stale):   # nothing of the other flag set survives, even if this build fails half-way
                os.remove(stale)
        with open(stamp, "w") as f:
            f.write(flags_now)
    todo = []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(OBJ, s[:-3] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr, os.path.getmtime(src)):
            todo.append((src, obj))
    objs = [os.path.join(OBJ, s[:-3] + ".o") for s in SOURCES]
    if not todo and os.path.exists(OUT) and os.path.getmtime(OUT) >= max(os.path.getmtime(o) for o in objs):
        return OUT
    outputs = []
    with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 1) or 1) as ex:
        for src, rc, out in ex.map(lambda so: _compile(nvcc, so[0], so[1], verbose, list(extra_flags)), todo):
            outputs.append("==== %s (rc %d)\n%s" % (os.path.basename(src), rc, out))
            if rc != 0:
                if log:
                    with open(log, "w") as f:
                        f.write("\n".join(outputs))
                raise RuntimeError("nvcc failed on %s:\n%s" % (src, out[-4000:]))
    if log:
        with open(log, "w") as f:
            f.write("\n".join(outputs))
    subprocess.check_call([nvcc, "-shared", "-o", OUT] + objs, cwd=HERE)
    return OUT


if __name__ == "__main__":
    flags = [a for a in sys.argv[1:] if a.startswith("-D")]
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, extra_flags=flags,
                log=os.environ.get("BCF_BUILD_LOG")))
