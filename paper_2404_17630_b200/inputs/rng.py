"""Counter-based hash RNG shared by every input generator (numpy, C++ and CUDA).

u01(seed, stream, index) is a pure function, so the Python, host C++ and device
generators produce identical bits for the same (seed, stream, index).
It holds none of the method's arithmetic: inputs only.

    mix(z):  z += 0x9E3779B97F4A7C15
             z  = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9
             z  = (z ^ (z >> 27)) * 0x94D049BB133111EB
             return z ^ (z >> 31)                       (splitmix64 finaliser)
    u01 = (mix(mix(seed + stream * 0x632BE59BD9B4E019) ^ index) >> 11) * 2^-53

The same three lines are restated in csrc/meshgen.cu (`mg_mix`, `mg_u01`).
"""
import numpy as np

_M1 = np.uint64(0x9E3779B97F4A7C15)
_M2 = np.uint64(0xBF58476D1CE4E5B9)
_M3 = np.uint64(0x94D049BB133111EB)
_MS = np.uint64(0x632BE59BD9B4E019)


def mix(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = z + _M1
        z = (z ^ (z >> np.uint64(30))) * _M2
        z = (z ^ (z >> np.uint64(27))) * _M3
        return z ^ (z >> np.uint64(31))


def u01(seed, stream, index):
    """Uniform doubles in [0,1) for an array of integer indices."""
    index = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        base = mix(np.uint64(seed) + np.uint64(stream) * _MS)
    z = mix(base ^ index)
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def normal(seed, stream, index):
    """Unit-variance Gaussian deviates (Box-Muller on two hash streams)."""
    u1 = u01(seed, 2 * stream, index)
    u2 = u01(seed, 2 * stream + 1, index)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)
