"""CPU ORACLE for the lost-sample normalisation -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu legs may import this.  Plain numpy and
Python loops, shares nothing with the CUDA path.  It follows PAPER.md section II-C ("GPU Post-Processing",
PAPER.md:111-121) step by step, in the paper's order:

  "Loss of input samples can result from packet loss, or numerical range and sampling limitations in the
   FPGAs and ADCs.  When this happens the data points are zeroed, before they are transferred to the GPU.
   This causes some correlated data points to contain fewer input samples in each integration."  (:113)

  1. "Packet loss is tracked as a single counter, then added to every point in the normalization matrix at
     the end of each integration."                                                                 (:115)
  2. "The F-engine flags are extracted from bit-fields in the packet footers and stored in counters for each
     input and frequency per integration.  The counters are used to populate the normalization matrix at the
     end of each integration."                                                                       (:116)
  3. "If two or more inputs are flaged by the F-engine in the same time sample, the previous step will result
     in a double counting in the normalization matrix at their intersections.  To correct this, these
     intersections are recorded per sample, and subtracted from the normalization matrix."       (:117-119)
  4. "The fraction of lost data given by the normalization matrix is then applied to the correlation
     matrix."                                                                                        (:121)

Readings where the paper is silent (N1..N5):
  N1  one flag bit per (time sample, channel, input); a flagged sample's voltage byte is zero in the frame.
  N2  the packet-loss counter is kept per frequency channel (lost[f] = time samples of channel f that were lost
      with their packets; a stream's counter applies to its 8 channels); a lost packet carries no flags.
  N3  step 2 "populate": counter c_f[n] is added to every point of row n and of column n of channel f's
      matrix; the autocorrelation point (n, n) lies in both and receives it once.
  N4  step 4 "applied": V~[i,j] = V[i,j] * T / (T - L[i,j]) with T the samples integrated since the last read,
      i.e. the sum is scaled to what T valid samples would have given; 0 where no valid sample is left.
  N5  the normalised visibilities are floating point (the paper does not say); the oracle computes in float64.

Pins (tests/test_oracle_normalisation.py): L equals T minus a direct count of the samples in which both inputs
were present (brute force over every pair and sample); hand-worked example (tests/golden/normalisation.txt);
no flags and no loss -> L = 0 and V~ = V; constant voltages with flagged samples zeroed -> V~ = T |c|^2 exactly.
"""
from __future__ import annotations

import numpy as np


def n_pairs(n_inputs: int) -> int:
    return n_inputs * (n_inputs + 1) // 2


def pair_index(n_inputs: int, i: int, j: int) -> int:
    """p(i,j) = i(2N-i+1)/2 + (j-i), i <= j (R4)."""
    return i * (2 * n_inputs - i + 1) // 2 + (j - i)


def flag_counters(flags: np.ndarray) -> np.ndarray:
    """Step 2, first half: counters for each input and frequency.  flags: bool[T][F][N] -> int64[F][N]."""
    flags = np.asarray(flags, dtype=bool)
    return flags.sum(axis=0, dtype=np.int64)


def flag_intersections(flags: np.ndarray) -> np.ndarray:
    """Step 3: intersections recorded per sample.  -> int64[F][P]; entry p(i,j), i < j, counts the time samples
    in which inputs i and j were both flagged (autocorrelation entries stay 0).  O(E^2) per sample, as in the paper."""
    flags = np.asarray(flags, dtype=bool)
    n_time, n_freq, n = flags.shape
    out = np.zeros((n_freq, n_pairs(n)), dtype=np.int64)
    for t in range(n_time):
        for f in range(n_freq):
            hit = np.flatnonzero(flags[t, f])
            for a in range(len(hit)):
                for b in range(a + 1, len(hit)):
                    out[f, pair_index(n, int(hit[a]), int(hit[b]))] += 1
    return out


def lost_matrix(flags: np.ndarray, lost: np.ndarray) -> np.ndarray:
    """The normalisation matrix L[f][p(i,j)] built in the paper's order (steps 1-3).  lost: int[F] (N2)."""
    flags = np.asarray(flags, dtype=bool)
    n_time, n_freq, n = flags.shape
    lost = np.asarray(lost, dtype=np.int64).reshape(n_freq)
    L = np.zeros((n_freq, n_pairs(n)), dtype=np.int64)
    # 1. packet loss: a single counter added to every point
    L += lost[:, None]
    # 2. per-(input, frequency) flag counters populate row n and column n (N3: the point (n, n) once)
    c = flag_counters(flags)
    for f in range(n_freq):
        for k in range(n):
            if c[f, k] == 0:
                continue
            for j in range(k, n):          # row k: points (k, j), j >= k
                L[f, pair_index(n, k, j)] += c[f, k]
            for i in range(0, k):          # column k: points (i, k), i < k
                L[f, pair_index(n, i, k)] += c[f, k]
    # 3. subtract the double counting at the intersections
    L -= flag_intersections(flags)
    return L


def normalise(vis: np.ndarray, n_samples: int, L: np.ndarray) -> np.ndarray:
    """Step 4 (N4, N5): vis int[F][P][2], L int[F][P] -> float64[F][P][2] = V * T / (T - L); 0 where T - L <= 0."""
    vis = np.asarray(vis).astype(np.float64)
    valid = (np.int64(n_samples) - np.asarray(L, dtype=np.int64)).astype(np.float64)
    scale = np.where(valid > 0, np.float64(n_samples) / np.where(valid > 0, valid, 1.0), 0.0)
    return vis * scale[:, :, None]
