"""Seeded synthetic input generators shared by the oracle-side tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic: it only draws random voltages, quantises them to
4 bits and packs them into the wire format.  Bytes are generated once on the host and the identical
buffer is handed to both the oracle and the CUDA path, so generator rounding can never cause a mismatch.

Wire format (nibble order and sign from BASELINE.json:north_star (a)):
one byte per (t, f, input) sample, ``byte = ((re & 15) << 4) | (im & 15)``, re/im signed 4-bit two's
complement in [-8, 7]; frame layout ``uint8[T][F][N]`` with the input index fastest.

The inputs stand in for the paper's live telescope stream; recipes follow
BASELINE.json:configs and SURVEY.md section 8(d) (restated in DESIGN.md "Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


def pack(re: np.ndarray, im: np.ndarray) -> np.ndarray:
    """Pack integer re/im in [-8, 7] into wire bytes (re -> high nibble, im -> low nibble)."""
    re = np.asarray(re).astype(np.int16)
    im = np.asarray(im).astype(np.int16)
    if re.min(initial=0) < -8 or re.max(initial=0) > 7 or im.min(initial=0) < -8 or im.max(initial=0) > 7:
        raise ValueError("re/im outside [-8, 7]")
    return (((re & 15) << 4) | (im & 15)).astype(np.uint8)


def _quantise(x: np.ndarray) -> np.ndarray:
    """Round half to even, clip to [-8, 7] (tails fold into -8 and 7)."""
    return np.clip(np.rint(x), -8, 7).astype(np.int8)


def uniform_frame(n_inputs: int, n_freq: int, n_time: int, seed: int) -> np.ndarray:
    """Every byte uniform on 0..255  <=>  re, im independent uniform on [-8, 7] (config C1)."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, 256, size=(n_time, n_freq, n_inputs), dtype=np.uint8)


def gaussian_frame(n_inputs: int, n_freq: int, n_time: int, seed: int, sigma: float = 2.5,
                   sigma_sky: float = 0.0, t_chunk: int | None = None) -> np.ndarray:
    """re, im = clip(rint(N(0, sigma^2)), -8, 7) independently per (t, f, n) (configs C2, C3).

    With ``sigma_sky`` > 0 one shared complex Gaussian s(t, f) with re, im ~ N(0, sigma_sky^2) is added
    to all inputs *before* quantisation (config C4), so off-diagonal visibilities have nonzero mean.
    Generated in chunks of time samples from one seeded stream, so the result depends only on
    (shape, seed, sigma, sigma_sky, t_chunk).
    """
    rng = np.random.default_rng(seed)
    out = np.empty((n_time, n_freq, n_inputs), dtype=np.uint8)
    if t_chunk is None:
        t_chunk = max(1, (1 << 24) // max(1, n_freq * n_inputs))
    for t0 in range(0, n_time, t_chunk):
        t1 = min(n_time, t0 + t_chunk)
        shape = (t1 - t0, n_freq, n_inputs)
        re = rng.standard_normal(shape, dtype=np.float32) * np.float32(sigma)
        im = rng.standard_normal(shape, dtype=np.float32) * np.float32(sigma)
        if sigma_sky > 0.0:
            sky = rng.standard_normal((2, t1 - t0, n_freq, 1), dtype=np.float32) * np.float32(sigma_sky)
            re += sky[0]
            im += sky[1]
        qr = _quantise(re).view(np.uint8)
        qi = _quantise(im).view(np.uint8)
        out[t0:t1] = ((qr & 15) << 4) | (qi & 15)
    return out


def stress_frame(n_inputs: int, n_freq: int, n_time: int, seed: int) -> np.ndarray:
    """First half of the inputs fixed at -8-8j (byte 0x88), second half uniform bytes (config C5)."""
    rng = np.random.default_rng(seed)
    out = np.empty((n_time, n_freq, n_inputs), dtype=np.uint8)
    half = n_inputs // 2
    out[:, :, :half] = 0x88
    t_chunk = max(1, (1 << 26) // max(1, n_freq * n_inputs))
    for t0 in range(0, n_time, t_chunk):
        t1 = min(n_time, t0 + t_chunk)
        out[t0:t1, :, half:] = rng.integers(0, 256, size=(t1 - t0, n_freq, n_inputs - half), dtype=np.uint8)
    return out


def constant_frame(n_inputs: int, n_freq: int, n_time: int, byte: int) -> np.ndarray:
    return np.full((n_time, n_freq, n_inputs), byte, dtype=np.uint8)


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: shape, generator, seed."""
    name: str
    n_inputs: int
    n_freq: int
    n_time: int
    kind: str           # "uniform" | "gaussian" | "gaussian_sky" | "stress"
    seed: int
    n_frames: int = 1   # C3 streams 64 frames; frame k uses seed + k
    note: str = ""

    @property
    def frame_bytes(self) -> int:
        return self.n_inputs * self.n_freq * self.n_time

    @property
    def n_pairs(self) -> int:
        return self.n_inputs * (self.n_inputs + 1) // 2

    @property
    def output_bytes(self) -> int:
        return self.n_freq * self.n_pairs * 8

    @property
    def cmacs_per_frame(self) -> int:
        return self.n_freq * self.n_time * self.n_pairs

    def frame(self, k: int = 0, n_time: int | None = None) -> np.ndarray:
        """Frame k of this config (optionally with fewer time samples, same stream prefix not implied)."""
        t = self.n_time if n_time is None else n_time
        return make_frame(self.kind, self.n_inputs, self.n_freq, t, self.seed + k)


def make_frame(kind: str, n_inputs: int, n_freq: int, n_time: int, seed: int) -> np.ndarray:
    if kind == "uniform":
        return uniform_frame(n_inputs, n_freq, n_time, seed)
    if kind == "gaussian":
        return gaussian_frame(n_inputs, n_freq, n_time, seed)
    if kind == "gaussian_sky":
        return gaussian_frame(n_inputs, n_freq, n_time, seed, sigma_sky=1.0)
    if kind == "stress":
        return stress_frame(n_inputs, n_freq, n_time, seed)
    raise ValueError(f"unknown kind {kind!r}")


# BASELINE.json:configs[0..4]  (seeds: C1's is given; the others are this build's)
CONFIGS = {
    "C1": Config("C1", 16, 4, 256, "uniform", 0, note="tiny correctness"),
    "C2": Config("C2", 256, 64, 16384, "gaussian", 2, note="CHIME Pathfinder per-server frame, 256 MiB"),
    "C3": Config("C3", 256, 1024, 4096, "gaussian", 3000, n_frames=64, note="full band streamed, 1 GiB frames"),
    "C4": Config("C4", 2048, 16, 8192, "gaussian_sky", 4, note="larger-N scaling, common sky signal"),
    "C5": Config("C5", 512, 32, 131072, "stress", 5, note="saturation / overflow stress, 2 GiB"),
}


# ----------------------------------------------------------------------------------------------------------
# F-engine flags and packet loss (NEXT-1; NEXT-2).  Only draws and packs: the
# normalisation arithmetic lives in the CUDA path and, separately, in oracle/normalisation.py.
# ----------------------------------------------------------------------------------------------------------
PACKET_T = 4      # time samples per UDP packet
PACKET_F = 8      # frequency channels per 10 GbE stream / packet


def pack_flags(flags: np.ndarray) -> np.ndarray:
    """bool[T][F][N] -> wire bit-field uint8[T][F][N/8]: input n is bit (n % 8) of byte n // 8 (N1)."""
    flags = np.asarray(flags, dtype=bool)
    if flags.shape[-1] % 8:
        raise ValueError("N must be a multiple of 8")
    return np.packbits(flags, axis=-1, bitorder="little")


def draw_flags_and_loss(n_inputs: int, n_freq: int, n_time: int, seed: int, p_flag: float = 1e-3, p_burst: float = 2e-4,
                        burst_frac: float = 0.05, p_packet_loss: float = 2e-3):
    """Seeded F-engine flags and packet loss for one frame.

    * each (t, f, n) sample is flagged independently with probability p_flag (ADC / FFT range errors);
    * with probability p_burst a whole (t, f) sample has a further burst_frac of its inputs flagged at once
      (several inputs flagged in the same time sample: the paper's intersections);
    * packets of PACKET_T samples x PACKET_F channels x all inputs are lost with probability p_packet_loss; a lost
      packet carries no flags (its footer never arrived).
    Returns flags bool[T][F][N], lost_mask bool[T][F], lost int32[F] (lost time samples per channel).
    The paper gives no rates ("provided E << N"); these are this build's.
    """
    rng = np.random.default_rng(seed)
    flags = rng.random((n_time, n_freq, n_inputs), dtype=np.float32) < np.float32(p_flag)
    burst = rng.random((n_time, n_freq)) < p_burst
    for t, f in zip(*np.nonzero(burst)):
        flags[t, f] |= rng.random(n_inputs) < burst_frac
    npt, npf = -(-n_time // PACKET_T), -(-n_freq // PACKET_F)
    lost_pkt = rng.random((npt, npf)) < p_packet_loss
    lost_mask = np.repeat(np.repeat(lost_pkt, PACKET_T, axis=0), PACKET_F, axis=1)[:n_time, :n_freq]
    flags &= ~lost_mask[:, :, None]
    lost = lost_mask.sum(axis=0).astype(np.int32)
    return flags, lost_mask, lost


def zero_lost_samples(frame: np.ndarray, flags: np.ndarray, lost_mask: np.ndarray) -> np.ndarray:
    """"When this happens the data points are zeroed, before they are transferred to the GPU"."""
    out = frame.copy()
    out[flags] = 0
    out[lost_mask] = 0
    return out
