"""Counter-based random numbers for the synthetic inputs.

A stateless 64-bit mix (splitmix64 finaliser) of (seed, stream, index, dim)
gives a uniform double in [0, 1).  Everything is vectorised numpy on uint64
with wrap-around arithmetic, so one value never depends on how many others were
drawn: the same (seed, stream, index, dim) always gives the same number.

This module belongs to the input generators only.  It holds none of the
method's arithmetic and is the one piece of code the oracle's tests and the
CUDA path's tests both consume (through the arrays it produces).
"""
import numpy as np

_U = np.uint64
_GOLD = _U(0x9E3779B97F4A7C15)
_M1 = _U(0xBF58476D1CE4E5B9)
_M2 = _U(0x94D049BB133111EB)
_K_IDX = _U(0xD1B54A32D192ED03)
_K_DIM = _U(0x8CB92BA72F3D8DD7)


def _mix64(z):
    z = (z ^ (z >> _U(30))) * _M1
    z = (z ^ (z >> _U(27))) * _M2
    return z ^ (z >> _U(31))


def hash_u64(seed, stream, index, dim):
    """uint64 hash; `index` and `dim` may be arrays (broadcast together)."""
    with np.errstate(over="ignore"):
        index = np.asarray(index, dtype=np.uint64)
        dim = np.asarray(dim, dtype=np.uint64)
        h = _mix64(_U(seed & 0xFFFFFFFFFFFFFFFF) + _GOLD * _U(stream + 1))
        h = _mix64(h ^ (index * _K_IDX))
        h = _mix64(h ^ (dim * _K_DIM + _GOLD))
    return h


def u01(seed, stream, index, dim):
    """Uniform float64 in [0, 1) with 53 random bits."""
    return (hash_u64(seed, stream, index, dim) >> _U(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(seed, stream, index, dim):
    """Standard normal via Box-Muller on two uniforms (dims 2*dim, 2*dim+1)."""
    dim = np.asarray(dim, dtype=np.uint64)
    u1 = u01(seed, stream, index, dim * _U(2))
    u2 = u01(seed, stream, index, dim * _U(2) + _U(1))
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)
