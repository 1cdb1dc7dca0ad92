"""Pins for oracle/normalisation.py (NEXT-1) -- CPU only.

The oracle builds the normalisation matrix the way the paper describes it (loss counter + flag counters -
per-sample intersections).  It is pinned to what that matrix must MEAN: L[i,j] = T - #{samples in which both
inputs were present}, counted here directly, pair by pair and sample by sample, without counters or
inclusion-exclusion; to the pencil-worked case in tests/golden/normalisation.txt; and, through the correlation
oracle, to the closed form "constant voltages with lost samples zeroed normalise back to T |c|^2".
"""
from pathlib import Path

import numpy as np
import pytest

import oracle
import workloads as wl
from oracle import normalisation as on

GOLDEN = Path(__file__).parent / "golden" / "normalisation.txt"


def valid_count_direct(flags, lost_mask):
    """#samples in which inputs i and j are both present, by definition (no counters, no inclusion-exclusion)."""
    t, f, n = flags.shape
    present = ~flags & ~lost_mask[:, :, None]
    out = np.zeros((f, on.n_pairs(n)), dtype=np.int64)
    for ch in range(f):
        for i in range(n):
            for j in range(i, n):
                cnt = 0
                for s in range(t):
                    if present[s, ch, i] and present[s, ch, j]:
                        cnt += 1
                out[ch, on.pair_index(n, i, j)] = cnt
    return out


def case_a():
    flags = np.zeros((4, 1, 16), dtype=bool)
    flags[0, 0, 1] = True
    flags[1, 0, 1] = True
    flags[1, 0, 3] = True
    lost_mask = np.zeros((4, 1), dtype=bool)
    lost_mask[3, 0] = True
    return flags, lost_mask, np.array([1], dtype=np.int32)


def test_handworked_case_a():
    flags, lost_mask, lost = case_a()
    L = on.lost_matrix(flags, lost)
    rows = [ln.split() for ln in GOLDEN.read_text().splitlines() if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 11
    for i, j, want_l, want_valid in rows:
        i, j = int(i), int(j)
        assert L[0, on.pair_index(16, i, j)] == int(want_l), (i, j)
        assert 4 - L[0, on.pair_index(16, i, j)] == int(want_valid), (i, j)
    # the normalised values of the golden file's last lines
    frame = wl.zero_lost_samples(wl.constant_frame(16, 1, 4, 0x30), flags, lost_mask)
    vis = oracle.naive(frame)
    assert vis[0, on.pair_index(16, 1, 3)].tolist() == [9, 0] and vis[0, 0].tolist() == [27, 0]
    vn = on.normalise(vis, 4, L)
    assert vn[0, on.pair_index(16, 1, 3)].tolist() == [36.0, 0.0]
    assert vn[0, 0].tolist() == [36.0, 0.0]


@pytest.mark.parametrize("n,f,t,seed", [(16, 2, 40, 1), (32, 3, 25, 2), (48, 1, 64, 3)])
def test_matrix_equals_direct_count_of_present_samples(n, f, t, seed):
    # dense flags and loss so that every branch (autos, intersections of 2 and more inputs, loss) is exercised
    flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, seed, p_flag=0.08, p_burst=0.1, burst_frac=0.3, p_packet_loss=0.15)
    assert flags.any() and lost.any() and (flags.sum(axis=2) >= 3).any()
    L = on.lost_matrix(flags, lost)
    assert np.array_equal(t - L, valid_count_direct(flags, lost_mask))


def test_counters_and_intersections_separately():
    flags = np.zeros((3, 2, 16), dtype=bool)
    flags[0, 1, [2, 5, 9]] = True
    flags[2, 1, [5, 9]] = True
    c = on.flag_counters(flags)
    assert c[1, 2] == 1 and c[1, 5] == 2 and c[1, 9] == 2 and c.sum() == 5 and c[0].sum() == 0
    x = on.flag_intersections(flags)
    assert x[1, on.pair_index(16, 2, 5)] == 1 and x[1, on.pair_index(16, 2, 9)] == 1 and x[1, on.pair_index(16, 5, 9)] == 2
    assert x.sum() == 4 and x[0].sum() == 0


def test_no_flags_no_loss_is_the_identity():
    flags = np.zeros((8, 2, 16), dtype=bool)
    L = on.lost_matrix(flags, np.zeros(2, dtype=np.int32))
    assert not L.any()
    vis = oracle.naive(wl.uniform_frame(16, 2, 8, 7))
    assert np.array_equal(on.normalise(vis, 8, L), vis.astype(np.float64))


def test_loss_only_scales_every_point_alike():
    L = on.lost_matrix(np.zeros((10, 2, 16), dtype=bool), np.array([2, 5]))
    assert (L[0] == 2).all() and (L[1] == 5).all()
    vis = np.ones((2, on.n_pairs(16), 2), dtype=np.int32) * 8
    vn = on.normalise(vis, 10, L)
    assert np.allclose(vn[0], 10.0) and np.allclose(vn[1], 16.0)


def test_all_samples_lost_gives_zero_not_nan():
    L = np.full((1, on.n_pairs(16)), 6)
    vn = on.normalise(np.zeros((1, on.n_pairs(16), 2), dtype=np.int32), 6, L)
    assert not vn.any() and np.isfinite(vn).all()


@pytest.mark.parametrize("byte", [0x30, 0x8F, 0x7E])
def test_constant_voltages_normalise_back_to_t_c2(byte):
    # closed form through the correlation oracle: zeroed samples remove exactly (T - valid) |c|^2 from every pair,
    # so V~ = T |c|^2 (+0i) wherever at least one valid sample is left
    n, f, t = 32, 2, 48
    flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, 11, p_flag=0.05, p_burst=0.05, burst_frac=0.2, p_packet_loss=0.1)
    frame = wl.zero_lost_samples(wl.constant_frame(n, f, t, byte), flags, lost_mask)
    vis = oracle.planar(frame)
    L = on.lost_matrix(flags, lost)
    vn = on.normalise(vis, t, L)
    re, im = oracle.unpack(np.array([[[byte]]], dtype=np.uint8))
    c2 = float(int(re.ravel()[0]) ** 2 + int(im.ravel()[0]) ** 2)
    ok = (t - L) > 0
    assert ok.any()
    assert np.allclose(vn[..., 0][ok], t * c2, rtol=1e-12) and not vn[..., 1].any()


def test_pack_flags_bit_order():
    flags = np.zeros((1, 1, 16), dtype=bool)
    flags[0, 0, [0, 9, 15]] = True
    assert wl.pack_flags(flags).ravel().tolist() == [0x01, 0x82]


def test_generator_zeroes_and_disjointness():
    n, f, t = 64, 16, 64
    flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, 5, p_flag=0.01, p_packet_loss=0.05)
    assert not (flags & lost_mask[:, :, None]).any()          # a lost packet carries no flags
    assert np.array_equal(lost, lost_mask.sum(axis=0))
    # loss comes in packets of 4 samples x 8 channels
    blk = lost_mask.reshape(t // 4, 4, f // 8, 8)
    assert (blk.all(axis=(1, 3)) | ~blk.any(axis=(1, 3))).all()
    fr = wl.zero_lost_samples(wl.uniform_frame(n, f, t, 1) | 1, flags, lost_mask)
    assert not fr[flags].any() and not fr[lost_mask].any() and fr[~flags & ~lost_mask[:, :, None]].all()
