"""Counter-based uniform numbers for the *input generators only*.

Deliberately NOT Philox: the propagation path draws from Philox4x32-10 (DESIGN.md
section 3), and the generators must share no arithmetic with it.  Here a uniform is a
SplitMix64 finaliser (Steele, Lea & Flood, OOPSLA 2014) applied to
``hash(seed, stream) + index``, so element ``i`` of any stream can be generated on
its own -- which is what lets a test build the inputs of a sampled id subset of a
1e8-photon workload without generating the other photons.
"""
import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_STREAM_MUL = np.uint64(0xD1342543DE82EF95)


def _splitmix64(x):
    """SplitMix64 output function on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = (x + _GOLDEN).astype(np.uint64)
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def raw64(seed, stream, index):
    """64 pseudo-random bits for (seed, stream, index); index may be an array."""
    index = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        base = _splitmix64(np.asarray([np.uint64(seed) ^ (np.uint64(stream) * _STREAM_MUL)],
                                      dtype=np.uint64))[0]
        return _splitmix64(base + index)


def uniform01(seed, stream, index):
    """float64 uniforms in [0, 1) with 53 random bits."""
    return (raw64(seed, stream, index) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)
