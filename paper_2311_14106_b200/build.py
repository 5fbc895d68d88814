"""In-tree build of libdmrgk.so (sm_100a only) with nvcc.

    python -m paper_2311_14106_b200.build [--force] [--verbose]

Every .cu under csrc/ is compiled to an object under _build/ and linked into
_build/libdmrgk.so.  nvcc cross-compiles without a GPU.  The built library is
git-ignored but travels to the GPU box with the repository snapshot; it carries
the hash of the sources it was built from (source_hash), which dmrgk.load()
checks against the sources beside it.
"""
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "_build")
LIB = os.path.join(OUT, "libdmrgk.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

VERSION_SOURCE = "structure.cu"      # holds dmrgk_version(); compiled with -DDMRGK_SOURCE_HASH

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-O3,-Wall,-Wno-unused-function", "-I", INCLUDE,
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def _read(path):
    with open(path, "rb") as f:
        return f.read()


def _headers():
    hdrs = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith(".h")]
    hdrs += [os.path.join(INCLUDE, f) for f in sorted(os.listdir(INCLUDE)) if f.endswith(".h")]
    return hdrs


def _flags_blob():
    # the include path is machine-specific (the repo travels between boxes): hash the flags without it
    return " ".join(f for f in NVCC_FLAGS if f != INCLUDE).encode()


def source_hash():
    """Identity of what libdmrgk.so is built from: sha256 over every csrc/*.cu, csrc/*.h, include/*.h
    (names and contents) and the nvcc flags, 16 hex digits.  Compiled into dmrgk_version(), compared
    by dmrgk.load() and printed by bench.py, so a stale binary cannot be loaded unnoticed (file
    mtimes mean nothing after a checkout or a copy to another box)."""
    h = hashlib.sha256(_flags_blob())
    for path in sources() + _headers():
        h.update(os.path.basename(path).encode())
        h.update(_read(path))
    return h.hexdigest()[:16]


KERNEL_SOURCES = ("heff_kernels.cu", "tasklist.cu", "internal.h")


def kernel_hash():
    """Identity of what decides the GEMM kernel's memory traffic (the kernel, the work-list builder, the
    shared structures): keys the rows of profiles/traffic.csv that bench.py may quote."""
    h = hashlib.sha256(_flags_blob())
    for name in KERNEL_SOURCES:
        h.update(_read(os.path.join(CSRC, name)))
    return h.hexdigest()[:12]


def _object_hash(src, global_hash):
    h = hashlib.sha256(_flags_blob())
    h.update(_read(src))
    for path in _headers():
        h.update(_read(path))
    if os.path.basename(src) == VERSION_SOURCE:
        h.update(global_hash.encode())
    return h.hexdigest()[:16]


def _stamp(path):
    try:
        with open(path + ".hash") as f:
            return f.read().strip()
    except OSError:
        return None


def built_hash():
    """The source hash libdmrgk.so was linked from (None if there is no library or no stamp)."""
    return _stamp(LIB) if os.path.exists(LIB) else None


def build(force=False, verbose=False):
    """Compile and link; returns the path of libdmrgk.so.  Raises on any compiler error.  An object is
    recompiled when the hash of its source, the headers and the flags differs from its stamp.

    Safe to call from several processes at once (every rank of a torchrun job, parallel test workers):
    the whole build runs under an exclusive lock on _build/.lock, so the later callers wait and then find
    the stamps up to date; objects and the library are written under temporary names and renamed into
    place, so a process that dlopens the library meanwhile sees the old file or the new one, never half."""
    import fcntl
    os.makedirs(OUT, exist_ok=True)
    with open(os.path.join(OUT, ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            return _build_locked(force, verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _write_stamp(path, value):
    tmp = f"{path}.hash.tmp{os.getpid()}"
    with open(tmp, "w") as f:
        f.write(value)
    os.replace(tmp, path + ".hash")


def _build_locked(force, verbose):
    nvcc = _nvcc()
    srcs = sources()
    ghash = source_hash()
    objs = [os.path.join(OUT, os.path.basename(s)[:-3] + ".o") for s in srcs]

    def compile_one(pair):
        src, obj = pair
        want = _object_hash(src, ghash)
        if not force and os.path.exists(obj) and _stamp(obj) == want:
            return None
        extra = [f'-DDMRGK_SOURCE_HASH="{ghash}"'] if os.path.basename(src) == VERSION_SOURCE else []
        tmp = f"{obj}.tmp{os.getpid()}.o"
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", tmp]
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            if os.path.exists(tmp):
                os.remove(tmp)
            raise RuntimeError(f"nvcc failed on {src}:\n{p.stdout}\n{p.stderr}")
        os.replace(tmp, obj)
        _write_stamp(obj, want)
        return p.stderr if verbose else "compiled"

    with ThreadPoolExecutor(max_workers=min(8, len(srcs))) as ex:
        logs = list(ex.map(compile_one, zip(srcs, objs)))
    if verbose:
        for s, lg in zip(srcs, logs):
            if lg:
                print(f"--- {os.path.basename(s)}\n{lg}")
    if force or any(logs) or built_hash() != ghash:
        tmp = f"{LIB}.tmp{os.getpid()}.so"
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            if os.path.exists(tmp):
                os.remove(tmp)
            raise RuntimeError(f"link failed:\n{p.stdout}\n{p.stderr}")
        os.replace(tmp, LIB)
        _write_stamp(LIB, ghash)
    return LIB


if __name__ == "__main__":
    path = build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(path)
