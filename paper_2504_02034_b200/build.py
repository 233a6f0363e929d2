"""Build libchim.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Staleness is decided by content, not by file times: `source_hash()` (sha256 over the sources, the headers, the flags and this
file) is compiled into the library (`chim_build_id()`), written beside it (`libchim.so.srchash`) and checked by `binding.lib()`
after loading -- a libchim.so left over from other sources is rebuilt here and refused there, whatever its mtime says."""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libchim.so")
STAMP = OUT + ".srchash"
SOURCES = ["chim_api.cu", "k_tables.cu", "k_events.cu", "k_events_fast.cu", "k_inject.cu", "k_grad.cu", "k_peaks.cu", "k_pcat_static.cu"]
HEADERS = ["chim_internal.cuh", os.path.join("..", "..", "include", "chim.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=true", "-Xptxas", "-v"]


def source_hash() -> str:
    h = hashlib.sha256()
    for f in SOURCES + HEADERS:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()[:32]


def needs_build() -> bool:
    if not (os.path.exists(OUT) and os.path.exists(STAMP)):
        return True
    with open(STAMP) as f:
        return f.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    sh = source_hash()
    cmd = [nvcc] + NVCC_FLAGS + [f'-DCHIM_BUILD_ID="{sh}"', "-o", OUT] + [os.path.join(CSRC, f) for f in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libchim.so")
    with open(STAMP, "w") as f:
        f.write(sh + "\n")
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
