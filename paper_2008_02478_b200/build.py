"""Build libborisdemag.so in-tree with nvcc for sm_100a.

    python -m paper_2008_02478_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the
tree to the GPU box.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libborisdemag.so")
# one translation unit per group of kernels, compiled in parallel and linked into one library
SOURCES = [os.path.join(CSRC, f) for f in ("boris_demag.cu", "tu_t2d.cu", "tu_y3.cu", "tu_xz_a.cu", "tu_xz_b.cu",
                                            "tu_xz_c.cu", "tu_plane_x.cu", "tu_plane_yz.cu", "tu_plane_yz16.cu", "tu_plane_yz8.cu", "tu_plane_yz64.cu", "boris_llg.cu", "microbench.cu", "boris_demag_f64.cu", "boris_demag_ml.cu", "boris_demag_noalloc.cu")]
OBJDIR = os.path.join(HERE, "build")
NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found")


def _deps():
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(ROOT, "include", "boris_demag.h"))
    deps.append(os.path.join(ROOT, "include", "boris_llg.h"))
    deps.append(os.path.join(ROOT, "include", "boris_micro.h"))
    deps.append(os.path.join(ROOT, "include", "boris_demag_f64.h"))
    deps.append(os.path.join(ROOT, "include", "boris_demag_ml.h"))
    deps.append(os.path.join(ROOT, "include", "boris_demag_noalloc.h"))
    return deps


def up_to_date():
    if not os.path.exists(OUT):
        return False
    t = os.path.getmtime(OUT)
    return all(os.path.getmtime(d) <= t for d in _deps())


def build(force=False, verbose=False):
    """Compile the CUDA library if it is missing or older than its sources.  Returns its path."""
    if not force and up_to_date():
        return OUT
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJDIR, exist_ok=True)
    nvcc = _nvcc()

    def compile_one(src):
        obj = os.path.join(OBJDIR, os.path.basename(src)[:-3] + ".o")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
        res = subprocess.run(cmd, capture_output=True, text=True)
        return obj, cmd, res

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        results = list(pool.map(compile_one, SOURCES))
    for obj, cmd, res in results:
        if verbose:
            sys.stderr.write(res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", OUT + ".tmp"] + [r[0] for r in results]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    os.replace(OUT + ".tmp", OUT)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
