"""Counter-based RNG shared by every consumer of the synthetic inputs.

SURVEY.md 8(d): "64-bit SplitMix-style hash of (seed, stream, index) -> two
uniforms -> Box-Muller normal".  Being counter-based, element `index` of
stream `stream` has the same value no matter how the array is chunked.
"""
import numpy as np

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_GOLD = np.uint64(0x9E3779B97F4A7C15)


def _mix(z):
    """SplitMix64 finaliser on a uint64 array (wrapping arithmetic)."""
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _hash(seed, stream, index, lane):
    with np.errstate(over="ignore"):
        idx = np.asarray(index, dtype=np.uint64)
        key = _mix(np.uint64(seed) * _GOLD + np.uint64(stream))
        z = _mix(key + idx * _GOLD)
        z = _mix(z + np.uint64(lane) * _M2 + _GOLD)
    return z


def uniforms(seed, stream, index, lane=0):
    """Uniform doubles in (0, 1): 53 random bits, offset by half an ulp."""
    z = _hash(seed, stream, index, lane)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normals(seed, stream, index, pair=0):
    """Standard normals by Box-Muller.

    `pair` = 0 gives the cosine branch, 1 the sine branch of the same two
    uniforms, so (normals(...,0), normals(...,1)) are independent N(0,1).
    """
    u1 = uniforms(seed, stream, index, lane=0)
    u2 = uniforms(seed, stream, index, lane=1)
    r = np.sqrt(-2.0 * np.log(u1))
    ang = 2.0 * np.pi * u2
    return r * (np.cos(ang) if pair == 0 else np.sin(ang))


# ----------------------------------------------------------------------------
# The same generator on a torch device (for the cells whose psi block is too
# large to draw with numpy in reasonable time).  int64 arithmetic wraps exactly
# like uint64; logical shifts are emulated by masking.  Values can differ from
# the numpy path in the last ulp (device log/cos/sin), so a consumer that needs
# identical inputs on both sides copies the generated tensor, it does not
# regenerate it.
# ----------------------------------------------------------------------------
def _s64(v):
    v = int(v) & 0xFFFFFFFFFFFFFFFF
    return v - (1 << 64) if v >= (1 << 63) else v


def _t_shr(z, s):
    return (z >> s) & ((1 << (64 - s)) - 1)


def _t_mix(z):
    z = (z ^ _t_shr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _t_shr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _t_shr(z, 31)


def torch_normals_pair(seed, stream, index):
    """index: int64 torch tensor; returns (n0, n1) float64 tensors = normals(..., pair=0/1)."""
    import torch
    with np.errstate(over="ignore"):
        key = int(_mix(np.uint64(seed) * _GOLD + np.uint64(stream)))
    z = _t_mix(index * _s64(0x9E3779B97F4A7C15) + _s64(key))
    us = []
    for lane in (0, 1):
        zz = _t_mix(z + _s64((lane * 0x94D049BB133111EB + 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF))
        us.append((_t_shr(zz, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0))
    r = torch.sqrt(-2.0 * torch.log(us[0]))
    ang = (2.0 * np.pi) * us[1]
    return r * torch.cos(ang), r * torch.sin(ang)
