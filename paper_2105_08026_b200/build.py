"""Build paper_2105_08026_b200/libcudahm.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

One translation unit per compiled-in model (csrc/inst_*.cu) plus the host side (cudahm.cu) and the probes (probe.cu),
compiled in parallel into build/*.o and linked into one shared library.
"""
import concurrent.futures
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcudahm.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-cudart", "shared"]


def sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _inputs():
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    files += [os.path.join(ROOT, "include", f) for f in os.listdir(os.path.join(ROOT, "include"))]
    return files


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _inputs())


def _compile(nvcc, src, verbose, defines):
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    cmd = [nvcc] + NVCC_FLAGS + defines + ["-I" + os.path.join(ROOT, "include"), "-c", os.path.join(CSRC, src), "-o", obj]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    out = subprocess.run(cmd, cwd=HERE, capture_output=True, text=True)
    return src, obj, out.returncode, out.stdout + out.stderr


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        os.makedirs(OBJ, exist_ok=True)
        srcs = sources()
        objs, log = [], []
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(srcs), os.cpu_count() or 1)) as ex:
            for src, obj, rc, text in ex.map(lambda s: _compile(nvcc, s, verbose, list(defines)), srcs):
                log.append(f"== {src}\n{text}")
                if rc != 0:
                    raise RuntimeError(f"nvcc failed on {src}:\n{text}")
                objs.append(obj)
        if verbose:
            print("\n".join(log))
        subprocess.run([nvcc, "-shared", "-cudart", "shared", "-o", LIB] + objs, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
