"""Counter-based 64-bit generator (SplitMix64 finaliser) so every draw is a pure function of
(seed, counter) and inputs are reproducible on any machine and in any evaluation order."""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(x):
    """SplitMix64 output function applied to uint64 array ``x`` (wraps mod 2**64)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def keyed(seed, stream, counter):
    """uint64 hash of (seed, stream, counter); ``counter`` may be an array."""
    counter = np.asarray(counter, dtype=np.uint64)
    with np.errstate(over="ignore"):
        k = splitmix64(np.uint64(seed) ^ splitmix64(np.uint64(stream) * np.uint64(0xD6E8FEB86659FD93)))
        return splitmix64(k ^ splitmix64(counter))


def uniform_u53(seed, stream, counter):
    """Uniform doubles in [0, 1) with 53 random bits."""
    return (keyed(seed, stream, counter) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform_int(seed, stream, counter, lo, hi):
    """Uniform integers in [lo, hi] (inclusive), int64."""
    span = int(hi) - int(lo) + 1
    u = uniform_u53(seed, stream, counter)
    return (np.floor(u * span).astype(np.int64) + int(lo)).clip(lo, hi)


def normal(seed, stream, counter):
    """Standard normals via Box-Muller from two keyed uniforms."""
    counter = np.asarray(counter, dtype=np.uint64)
    u1 = uniform_u53(seed, stream, counter * np.uint64(2))
    u2 = uniform_u53(seed, stream, counter * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)
