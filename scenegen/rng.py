"""Counter-based SplitMix64 -> uniform doubles.  Own implementation so the streams are
bit-reproducible everywhere.  Value i of stream s of seed k is a pure
function of (k, s, i), so draws are vectorised with numpy uint64 wrap-around arithmetic."""
import numpy as np

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


class SplitMix:
    """A family of independent streams derived from one integer seed."""

    def __init__(self, seed: int):
        self.seed = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)
        self._next_stream = 0

    def _stream_key(self, stream: int) -> np.uint64:
        with np.errstate(over="ignore"):
            s = np.uint64(stream + 1) * np.uint64(0xD1342543DE82EF95)
            return _mix(np.array([self.seed ^ s], dtype=np.uint64))[0]

    def u64(self, n: int, stream: int = None) -> np.ndarray:
        if stream is None:
            stream = self._next_stream
            self._next_stream += 1
        key = self._stream_key(stream)
        i = np.arange(1, n + 1, dtype=np.uint64)
        with np.errstate(over="ignore"):
            return _mix(key + i * _GOLD)

    def uniform(self, n: int, lo: float = 0.0, hi: float = 1.0, stream: int = None) -> np.ndarray:
        """n doubles uniform in [lo, hi)."""
        u = (self.u64(n, stream) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        return lo + (hi - lo) * u

    def normal(self, n: int, stream: int = None) -> np.ndarray:
        """n standard normals (Box-Muller on two uniform streams)."""
        if stream is None:
            s1 = self._next_stream
            self._next_stream += 2
        else:
            s1 = stream
        u1 = self.uniform(n, stream=s1)
        u2 = self.uniform(n, stream=s1 + 1)
        r = np.sqrt(-2.0 * np.log(1.0 - u1))  # 1-u1 in (0,1]
        return r * np.cos(2.0 * np.pi * u2)
