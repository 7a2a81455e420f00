"""Seeded synthetic inputs for the FDAS hot path.

This module is the ONE piece of code that serves both the CUDA path and the CPU
oracle: it only manufactures input time series (noise + injected accelerated
sinusoids, BASELINE.json configs[0..4], reading G19). It holds
none of the method's arithmetic (no FFT, no templates, no correlation) and
imports neither `oracle/` nor the CUDA binding.

Random numbers come from an own counter-based generator (splitmix64 of
(seed, counter) -> two uniforms -> Box-Muller in fp64 -> float32), so the bits
do not depend on the numpy / torch version.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

BASE_SEED = 151107343

_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def splitmix64(x: np.ndarray) -> np.ndarray:
    """The splitmix64 finaliser applied element-wise to uint64 `x`."""
    with np.errstate(over="ignore"):
        z = (x + _GOLDEN).astype(_U64)
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        return z ^ (z >> _U64(31))


def _hash2(seed: int, counter: np.ndarray, lane: int) -> np.ndarray:
    """64 random bits for (seed, counter, lane)."""
    with np.errstate(over="ignore"):
        s = splitmix64(np.asarray([seed], dtype=_U64) * _U64(2) + _U64(lane))
        return splitmix64(counter.astype(_U64) ^ s)


def uniform01(seed: int, counter: np.ndarray, lane: int = 0) -> np.ndarray:
    """Uniform doubles in (0, 1): the top 53 bits of the hash, offset by half an ulp."""
    bits = _hash2(seed, counter, lane) >> _U64(11)
    return (bits.astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal_f64(seed: int, n: int, start: int = 0) -> np.ndarray:
    """n standard normals (fp64), samples start..start+n-1 of stream `seed`.

    Sample k uses counter k//2 and the cos (k even) or sin (k odd) Box-Muller branch.
    """
    k = np.arange(start, start + n, dtype=np.int64)
    c = (k >> 1).astype(_U64)
    u1 = uniform01(seed, c, 0)
    u2 = uniform01(seed, c, 1)
    r = np.sqrt(-2.0 * np.log(u1))
    ang = 2.0 * np.pi * u2
    return np.where((k & 1) == 0, r * np.cos(ang), r * np.sin(ang))


@dataclass
class Signal:
    """One injected accelerated sinusoid: A*cos(2*pi*[(r0 - z/2)*u + (z/2)*u^2] + phi), u = n/N.

    r0 is the MEAN (mid-span) Fourier frequency in bins, z the number of bins
    drifted over the span (reading G2/G5 of SURVEY.md §8(c))."""
    amp: float
    r0: float
    z: float
    phi: float = 0.0


def pulse_train(amp: float, r0: float, z0: float, n_harm: int, decay: float = 1.0, phi: float = 0.0):
    """The first `n_harm` harmonics of an accelerated pulsar: harmonic h sits at (h r0, h z0) with amplitude
    amp * decay^(h-1) ("pulse harmonics"; z scales with the frequency)."""
    return [Signal(amp * decay ** (h - 1), h * r0, h * z0, phi * h) for h in range(1, n_harm + 1)]


def make_series(n_samples: int, seed: int, signals=(), noise: bool = True,
                chunk: int = 1 << 21) -> np.ndarray:
    """float32[n_samples] = N(0,1) noise (stream `seed`) + the given signals."""
    out = np.empty(n_samples, dtype=np.float32)
    for s in range(0, n_samples, chunk):
        e = min(n_samples, s + chunk)
        x = normal_f64(seed, e - s, s) if noise else np.zeros(e - s)
        if signals:
            u = np.arange(s, e, dtype=np.float64) / float(n_samples)
            for sg in signals:
                cyc = (sg.r0 - 0.5 * sg.z) * u + (0.5 * sg.z) * u * u
                cyc -= np.floor(cyc)
                x = x + sg.amp * np.cos(2.0 * np.pi * cyc + sg.phi)
        out[s:e] = x.astype(np.float32)
    return out


@dataclass
class Config:
    """One BASELINE.json config: plan parameters + the injected signals per DM trial."""
    name: str
    index: int
    n_samples: int
    z_max: float
    dz: float
    width: int
    seg_len: int
    interbin: int = 0
    n_dm: int = 1
    threshold: float = 20.0
    signals: list = field(default_factory=list)  # list (per DM) of list[Signal]

    @property
    def n_bins(self) -> int:
        return self.n_samples // 2

    @property
    def n_z(self) -> int:
        return int(round(2 * self.z_max / self.dz)) + 1

    def series_seed(self, dm: int = 0) -> int:
        return BASE_SEED + 1000 * self.index + dm

    def series(self, dm: int = 0, noise: bool = True) -> np.ndarray:
        return make_series(self.n_samples, self.series_seed(dm), self.signals[dm], noise)


def _param_uniforms(index: int, n: int) -> np.ndarray:
    return uniform01(BASE_SEED + 7 * index, np.arange(n, dtype=np.uint64), 2)


def config(index: int, n_dm: int | None = None) -> Config:
    """BASELINE.json configs[index] with the G19 readings.

    Config 4 (harmonic sum) takes the config-2 series; its input plane is made from it.
    `n_dm` overrides the batch size of config 3 (64) for small parity cases."""
    if index == 0:
        return Config("tiny", 0, 1 << 17, 20.0, 2.0, 64, 1024, 0, 1, 20.0,
                      [[Signal(0.05, 10000.3, 8.0, 0.0)]])
    if index == 1:
        u = _param_uniforms(1, 16)
        sig = [Signal(0.02 + 0.03 * u[4 * i], 1e4 + (4e5 - 1e4) * u[4 * i + 1],
                      -90.0 + 180.0 * u[4 * i + 2], 2 * np.pi * u[4 * i + 3]) for i in range(4)]
        return Config("mid", 1, 1 << 20, 100.0, 2.0, 256, 2048, 1, 1, 20.0, [sig])
    if index in (2, 4):
        u = _param_uniforms(2, 32)
        sig = [Signal(0.01 + 0.02 * u[4 * i], 1e4 + (4e6 - 1e4) * u[4 * i + 1],
                      -80.0 + 160.0 * u[4 * i + 2], 2 * np.pi * u[4 * i + 3]) for i in range(8)]
        c = Config("ska" if index == 2 else "harmsum", 2, 1 << 23, 84.0, 2.0, 256, 2048, 0, 1, 20.0, [sig])
        return c
    if index == 3:
        nd = 64 if n_dm is None else n_dm
        n_sig = max(1, int(round(0.1 * nd)))
        u = _param_uniforms(3, 4 * 64 + 64)
        # seeded permutation of the DM indices: the first n_sig carry a signal
        order = np.argsort(u[256:256 + nd], kind="stable")
        sigs = [[] for _ in range(nd)]
        for i in range(n_sig):
            dm = int(order[i])
            sigs[dm] = [Signal(0.02, 1e4 + (4e6 - 1e4) * u[4 * i + 1],
                               -80.0 + 160.0 * u[4 * i + 2], 2 * np.pi * u[4 * i + 3])]
        return Config("batch", 3, 1 << 23, 84.0, 2.0, 256, 2048, 0, nd, 20.0, sigs)
    raise ValueError("config index must be 0..4")


def small_config(n_samples: int, z_max: float, dz: float, width: int, seg_len: int,
                 interbin: int = 0, n_dm: int = 1, n_sig: int = 2, index: int = 9,
                 amp: float = 0.08) -> Config:
    """A reduced-size config of the same recipe (parity cases the oracle finishes in seconds)."""
    nb = n_samples // 2
    u = _param_uniforms(index, 4 * n_sig * n_dm + 4)
    sigs = []
    for d in range(n_dm):
        s = []
        for i in range(n_sig):
            b = 4 * (d * n_sig + i)
            s.append(Signal(amp * (0.5 + u[b]), 0.05 * nb + 0.9 * nb * u[b + 1],
                            -0.9 * z_max + 1.8 * z_max * u[b + 2], 2 * np.pi * u[b + 3]))
        sigs.append(s)
    return Config("small", index, n_samples, z_max, dz, width, seg_len, interbin, n_dm, 20.0, sigs)
