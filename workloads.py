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


# ----------------------------------------------------------------------------------------------------------
# UDP packets (NEXT-2).  Formatting and shuffling only: the assembly itself lives in the CUDA
# path and, separately, in oracle/assembly.py.  Wire format = DESIGN.md section 13, reading P1.
# ----------------------------------------------------------------------------------------------------------
PACKET_MAGIC = 0x58454E47
PACKET_HEADER_BYTES = 32


def packetise(frame: np.ndarray, flag_bits: np.ndarray, seq0: int, s_per_packet: int = PACKET_T,
              c_per_packet: int = PACKET_F) -> np.ndarray:
    """Cut frame uint8[T][F][N] and its flag bit-field uint8[T][F][N/8] into packets, time-major then stream.

    Returns uint8[n_packets][packet_bytes]: 32-byte header {u32 magic, u32 stream_id, u64 seq, 16 zero bytes},
    payload uint8[S][C][N], footer uint8[S][C][N/8] (little endian).
    """
    T, F, N = frame.shape
    S, C = s_per_packet, c_per_packet
    assert T % S == 0 and F % C == 0 and flag_bits.shape == (T, F, N // 8)
    nb, ns = T // S, F // C
    pay = frame.reshape(nb, S, ns, C, N).transpose(0, 2, 1, 3, 4).reshape(nb * ns, S * C * N)
    foot = flag_bits.reshape(nb, S, ns, C, N // 8).transpose(0, 2, 1, 3, 4).reshape(nb * ns, S * C * N // 8)
    hdr = np.zeros((nb * ns, PACKET_HEADER_BYTES), dtype=np.uint8)
    blk, stream = np.divmod(np.arange(nb * ns, dtype=np.uint64), np.uint64(ns))
    hdr[:, 0:4] = np.full(nb * ns, PACKET_MAGIC, dtype="<u4").view(np.uint8).reshape(-1, 4)
    hdr[:, 4:8] = stream.astype("<u4").view(np.uint8).reshape(-1, 4)
    hdr[:, 8:16] = (np.uint64(seq0) + blk * np.uint64(S)).astype("<u8").view(np.uint8).reshape(-1, 8)
    return np.ascontiguousarray(np.concatenate([hdr, pay, foot], axis=1))


def disturb_packets(packets: np.ndarray, seed: int, p_loss: float = 2e-3, p_dup: float = 1e-3, p_late: float = 5e-3,
                    max_delay: int = 40, n_foreign: int = 0) -> np.ndarray:
    """A UDP network's effect on an in-order packet sequence ("lost, out of order, and duplicate
    packets"): drop with p_loss, repeat with p_dup (the copy arrives a little later), delay with p_late by up to
    max_delay positions, and insert n_foreign packets that do not belong (bad magic / stream / sequence number).
    Returns the packets in ARRIVAL order, uint8[n_arrived][packet_bytes].
    """
    rng = np.random.default_rng(seed)
    n = packets.shape[0]
    keep = rng.random(n) >= p_loss
    order_key = np.arange(n, dtype=np.float64)
    late = rng.random(n) < p_late
    order_key = order_key + late * rng.integers(1, max_delay + 1, n)
    idx = np.nonzero(keep)[0]
    key = order_key[idx]
    dup = idx[rng.random(idx.size) < p_dup]
    idx = np.concatenate([idx, dup])
    key = np.concatenate([key, order_key[dup] + rng.integers(1, max_delay + 1, dup.size) + 0.5])
    arrived = packets[idx[np.argsort(key, kind="stable")]].copy()
    if n_foreign:
        extra = packets[rng.integers(0, n, n_foreign)].copy()
        for k in range(n_foreign):
            kind = k % 3
            if kind == 0:
                extra[k, 0] ^= 0xFF                                  # wrong magic
            elif kind == 1:
                extra[k, 4:8] = np.array([0xFF, 0xFF, 0, 0], np.uint8)   # stream_id out of range
            else:
                extra[k, 8:16] = np.frombuffer(np.uint64(2 ** 40 + 1 + k).tobytes(), np.uint8)   # far-away, misaligned seq
        pos = np.sort(rng.integers(0, arrived.shape[0] + 1, n_foreign))
        arrived = np.insert(arrived, pos, extra, axis=0)
    return np.ascontiguousarray(arrived)


def sparse_flag_bits(n_inputs: int, n_freq: int, n_time: int, seed: int, rate: float = 1e-4) -> np.ndarray:
    """Cheap flag bit-field uint8[T][F][N/8] for full-size runs: about `rate` of the bytes get a random non-zero value
    (1-8 inputs of one sample flagged together, E << N)."""
    rng = np.random.default_rng(seed)
    fb = np.zeros((n_time, n_freq, n_inputs // 8), dtype=np.uint8)
    hit = rng.integers(0, fb.size, max(1, int(fb.size * rate)))
    fb.reshape(-1)[hit] = rng.integers(1, 256, hit.size, dtype=np.uint8)
    return fb
