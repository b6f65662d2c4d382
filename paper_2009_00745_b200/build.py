"""Builds liblise.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
import fcntl
import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "liblise.so")
# source -> extra flags; happly_yz_whole.cu: the whole-state FFT yz kernels are faster with ptxas' lower register-usage
# level (fewer spills at their 168-register cap), every other kernel with the default (csrc/fft_plane_kernels.cuh)
# no_alloc.cu: the allocation-free entry point and its fixed device array live in one translation unit of their own
SOURCES = {"lise.cu": [], "happly_yz_whole.cu": ["-Xptxas", "--register-usage-level=3"], "no_alloc.cu": []}
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def _deps():
    return ([f for f in glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
             if not f.endswith("line_codelets.cuh")]
            + glob.glob(os.path.join(CSRC, "*.py")) + [os.path.join(HERE, "..", "include", "lise.h")])


def _codelets():
    """(re)generate csrc/line_codelets.cuh, the straight-line FFT code of the line operators, from gen_codelets.py"""
    gen = os.path.join(CSRC, "gen_codelets.py")
    out = os.path.join(CSRC, "line_codelets.cuh")
    if os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(gen):
        return
    import importlib.util
    spec = importlib.util.spec_from_file_location("lise_gen_codelets", gen)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.generate(out)


def needs_build():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force=False, verbose=False):
    """Compile under a file lock (several ranks may call this at once): nvcc writes a temporary file that is
    renamed over liblise.so, so no process can dlopen a partly written library."""
    if not force and not needs_build():
        return SO
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not needs_build():      # another process built it while we waited
                return SO
            _codelets()
            nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
            tmp = SO + f".tmp{os.getpid()}"
            objs, procs = [], []
            for src, extra in SOURCES.items():                # the translation units compile side by side
                obj = os.path.join(CSRC, src[:-3] + f".tmp{os.getpid()}.o")
                objs.append(obj)
                cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
                procs.append((cmd, subprocess.Popen(cmd, cwd=CSRC)))
            try:
                for cmd, p in procs:
                    if p.wait() != 0:
                        raise subprocess.CalledProcessError(p.returncode, cmd)
                subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs, check=True, cwd=CSRC)
                os.replace(tmp, SO)
            finally:
                for o in objs:
                    if os.path.exists(o):
                        os.unlink(o)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
