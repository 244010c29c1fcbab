"""Counter-based seeded random numbers for the synthetic workloads.

u(seed, stream, idx) = top 53 bits of a twice-SplitMix64-finalised mix of (seed, stream, idx).
Stateless, vectorised, reproducible on any machine; normals by Box-Muller on the pair
(2k, 2k+1).  Holds none of the method's arithmetic: it only draws inputs.
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_G = np.uint64(0x9E3779B97F4A7C15)
_A = np.uint64(0xBF58476D1CE4E5B9)
_B = np.uint64(0x94D049BB133111EB)

# one stream id per tensor so that changing one input never shifts another
STREAMS = dict(positions=1, species=2, W_r=3, V=4, path_w=5, q=6, G=7, mol_size=8, mol_parent=9,
               mol_dir=10, mol_bond=11, W_x0=12, W_v0=13, W_w=14, W_p=15, A_lat=16, sample=17, rot=18)


def _fin(z):
    z = (z + _G)
    z = (z ^ (z >> np.uint64(30))) * _A
    z = (z ^ (z >> np.uint64(27))) * _B
    return z ^ (z >> np.uint64(31))


def bits(seed, stream, idx):
    """uint64 hash of (seed, stream, idx); idx may be an array."""
    idx = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        base = _fin(np.uint64(seed) * _G + np.uint64(stream) * _A + np.uint64(0x632BE59BD9B4E019))
        z = _fin(base ^ (idx * _B + _G))
        z = _fin(z)
    return z


def uniform(seed, stream, idx):
    """float64 in [0, 1)"""
    return (bits(seed, stream, idx) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed, stream, shape, offset=0):
    """float64 N(0,1) array of the given shape; element k uses counters (2k, 2k+1)."""
    count = int(np.prod(shape)) if len(shape) else 1
    out = np.empty(count, dtype=np.float64)
    step = 1 << 22
    for s in range(0, count, step):
        k = np.arange(s, min(s + step, count), dtype=np.uint64) + np.uint64(offset)
        u1 = uniform(seed, stream, 2 * k)
        u2 = uniform(seed, stream, 2 * k + 1)
        out[s:s + k.shape[0]] = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)
    return out.reshape(shape)


def randint(seed, stream, idx, lo, hi):
    """integers uniform in [lo, hi] inclusive"""
    return lo + np.floor(uniform(seed, stream, idx) * (hi - lo + 1)).astype(np.int64)
