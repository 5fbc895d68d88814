"""Counter-based random stream, bit-identical on host (NumPy) and device (CUDA).

Every number is a pure function of (seed, stream id, element index), so any
block of any arena can be regenerated anywhere without generating the rest.

``normal12`` is the value distribution used for every "N(0,1)" entry of the
synthetic workloads (BASELINE.json configs 2-5): the classical sum of twelve
uniforms (Irwin-Hall), mean 0, variance 1 - 2**-64, support (-6, 6).  It uses
integer arithmetic only (twelve 32-bit uniforms summed exactly, one exact
power-of-two scaling), so the NumPy implementation here and the CUDA fill
kernel of the library (`dmrgk_fill_normal`, a harness kernel outside the hot
path) produce identical bits; a Box-Muller transform would differ in the last
ulp between libm and the device math library.  DESIGN.md records this reading.
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


def splitmix64(x):
    """SplitMix64 finaliser applied to ``x + golden``; uint64 in, uint64 out."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = x + _GOLD
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        z = z ^ (z >> np.uint64(31))
    return z


def stream_base(seed, stream):
    """Base counter of stream ``stream`` under ``seed``."""
    s = splitmix64(np.uint64(stream & 0xFFFFFFFFFFFFFFFF))
    return splitmix64(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) ^ s)


def uniform_u64(seed, stream, index):
    """One 64-bit uniform integer per element index."""
    base = stream_base(seed, stream)
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        return splitmix64(base + idx)


def normal12(seed, stream, index):
    """Unit-variance bell-shaped value for each element index (see module doc).

    x = (sum of twelve 32-bit uniforms - 6*(2**32 - 1)) / 2**32, the uniforms
    being the high and low halves of splitmix64(base + 6*index + j), j = 0..5.
    """
    base = stream_base(seed, stream)
    idx = np.asarray(index, dtype=np.uint64)
    acc = np.zeros(idx.shape, dtype=np.uint64)
    with np.errstate(over="ignore"):
        c0 = base + idx * np.uint64(6)
        for j in range(6):
            h = splitmix64(c0 + np.uint64(j))
            acc = acc + (h >> np.uint64(32)) + (h & np.uint64(0xFFFFFFFF))
    centred = acc.astype(np.int64) - np.int64(6 * (2 ** 32 - 1))
    return centred.astype(np.float64) * (1.0 / 4294967296.0)
