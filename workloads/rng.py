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


# ---------------------------------------------------------------------------------------------------
# The same generator with torch ops, so that the feature tensors of the full-size configs (up to 86 GB)
# can be drawn directly in device memory.  Integer hashing is bit-identical to bits() above (int64
# arithmetic wraps mod 2^64; logical shifts are emulated); the Box-Muller floating point may differ from
# numpy's in the last place, so whoever needs the exact values (the oracle) reads them back from the tensor.
def _s64(x):
    x = int(x) & 0xFFFFFFFFFFFFFFFF
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z, k):
    return (z >> k) & ((1 << (64 - k)) - 1)


def _fin_torch(z):
    z = z + _s64(_G)
    z = (z ^ _lsr(z, 30)) * _s64(_A)
    z = (z ^ _lsr(z, 27)) * _s64(_B)
    return z ^ _lsr(z, 31)


def bits_torch(seed, stream, idx):
    """idx: int64 tensor of non-negative counters -> int64 tensor holding the same 64 bits as bits()"""
    with np.errstate(over="ignore"):
        base = _fin(np.uint64(seed) * _G + np.uint64(stream) * _A + np.uint64(0x632BE59BD9B4E019))
    z = _fin_torch((idx * _s64(_B) + _s64(_G)) ^ _s64(base))
    return _fin_torch(z)


def uniform_torch(seed, stream, idx):
    import torch
    return _lsr(bits_torch(seed, stream, idx), 11).to(torch.float64) * (1.0 / 9007199254740992.0)


def normal_torch(seed, stream, shape, offset=0, device="cuda", dtype=None, chunk=1 << 24):
    """N(0,1) tensor of `shape` on `device`; element k uses counters (2k, 2k+1) like normal()."""
    import torch
    dtype = dtype or torch.float64
    count = int(np.prod(shape)) if len(shape) else 1
    out = torch.empty(count, dtype=dtype, device=device)
    for s in range(0, count, chunk):
        e = min(s + chunk, count)
        k = torch.arange(s + offset, e + offset, dtype=torch.int64, device=device)
        u1 = uniform_torch(seed, stream, 2 * k)
        u2 = uniform_torch(seed, stream, 2 * k + 1)
        out[s:e] = (torch.sqrt(-2.0 * torch.log(1.0 - u1)) * torch.cos(2.0 * np.pi * u2)).to(dtype)
    return out.reshape(shape)
