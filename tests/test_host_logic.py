"""Host-side work decomposition (csrc/schedule.hpp) -- CPU only, through xcorr_debug_schedule."""
import numpy as np
import pytest

import paper_1503_06189_b200 as xb
import workloads as wl

SHAPES = [(c.n_inputs, c.n_freq, c.n_time) for c in wl.CONFIGS.values()] + [
    (16, 1, 1), (48, 3, 31), (144, 3, 100), (208, 1, 33), (400, 2, 1000), (256, 7, 64), (512, 5, 65), (768, 2, 4096), (2048, 1, 64),
]


def _check(n, f, t, workers):
    seg, wb = xb.xcorr_debug_schedule(n, f, t, workers)
    kt = xb.xcorr_debug_stage_samples()
    n_stage = -(-t // kt)
    nb = -(-n // 256)
    nst = nb * (nb + 1) // 2
    assert wb[0] == 0 and wb[-1] == len(seg) and (np.diff(wb) >= 0).all()
    cover = np.zeros((f * nst, n_stage), dtype=np.int32)
    load = np.zeros(workers, dtype=np.int64)
    for w in range(workers):
        for k in range(wb[w], wb[w + 1]):
            ff, I, J, s0, s1, tile, slot = seg[k]
            assert 0 <= ff < f and 0 <= I <= J < nb and 0 <= s0 < s1 <= n_stage
            assert tile == ff * nst + I * (2 * nb - I + 1) // 2 + (J - I)
            cover[tile, s0:s1] += 1
            load[w] += (9 if I == J else 16) * (s1 - s0)
    assert (cover == 1).all(), "every (super-tile, stage) must be processed exactly once"
    # every segment owns its own accumulator slot; a tile's slots are contiguous and ordered by time
    assert sorted(seg[:, 6].tolist()) == list(range(len(seg)))
    order = np.lexsort((seg[:, 3], seg[:, 5]))
    assert (seg[order, 6] == np.arange(len(seg))).all()
    return load, n_stage


@pytest.mark.parametrize("n,f,t", SHAPES)
@pytest.mark.parametrize("workers", [74, 1, 7])
def test_schedule_covers_everything_once(n, f, t, workers):
    _check(n, f, t, workers)


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_schedule_is_balanced_on_the_benchmark_configs(name):
    c = wl.CONFIGS[name]
    load, n_stage = _check(c.n_inputs, c.n_freq, c.n_time, 74)
    mean = load.sum() / 74
    # water filling: no worker exceeds the mean by more than one whole item's worth of imbalance in the
    # data-parallel part (cost 16 vs 9 per stage) -- in practice within 2 %
    assert load.max() <= mean * 1.02 + 16, (load.max(), mean)


def test_bad_arguments():
    with pytest.raises(xb.XCorrError):
        xb.xcorr_debug_schedule(24, 1, 64, 74)
    with pytest.raises(xb.XCorrError):
        xb.xcorr_debug_schedule(16, 1, 64, 0)


# ------------------------------------------------------------------ bench.py arithmetic (no GPU: the functions are pure)
def _bench():
    import importlib
    return importlib.import_module("bench")


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_bench_issued_over_useful_counts_the_mmas_of_the_schedule(name):
    """issued / useful int8 ops: 2 MMAs of 2*256*256*32 ops per 32 samples on a diagonal super-tile, 4 above it, against
    8 ops per complex MAC of the pairs i <= j -- recounted here from the tile grid."""
    b = _bench()
    c = wl.CONFIGS[name]
    nb = -(-c.n_inputs // 256)
    issued_per_sample = (2 * nb + 4 * nb * (nb - 1) // 2) * (2 * 256 * 256 * 32) / 32
    useful_per_sample = 8 * c.n_pairs
    assert b.issued_over_useful(c) == pytest.approx(issued_per_sample / useful_per_sample, rel=1e-12)
    if c.n_inputs % 256 == 0:
        # whole super-tiles: a diagonal tile issues 2 * 65536 MACs for its 32896 useful pairs, an off-diagonal one 4 * 65536 for 65536
        assert 0.99 < b.issued_over_useful(c) <= 1.0


def test_bench_tensor_roofline_uses_the_measured_issue_ceiling():
    b = _bench()
    c = wl.CONFIGS["C2"]
    peaks = {"hbm_gbs": 6500.0, "bf16_burst": 1600.0, "bf16_sustained": 1400.0, "source": "test"}
    ceiling = {"burst_tops": 4400.0, "sustained_tops": 4500.0}
    k_ms = 0.1
    ops = 8.0 * c.n_freq * c.n_time * c.n_pairs
    r = b.tensor_roofline(c, k_ms, peaks, ceiling, "sustained")
    assert r["algorithmic_ops_per_launch"] == ops and r["achieved"] == pytest.approx(ops / 1e-4 / 1e12)
    assert r["peak"] == 4500.0 and r["frac"] == pytest.approx(r["achieved"] / 4500.0) and r["frac"] < 1.0
    assert r["frac_of_2x_bf16"] == pytest.approx(r["achieved"] / 2800.0)
    assert b.tensor_roofline(c, k_ms, peaks, ceiling, "burst")["peak"] == 4400.0
    # no probe in the run: the stand-in is 2 x the measured bf16 rate of the same leg, and the line says so
    r0 = b.tensor_roofline(c, k_ms, peaks, None, "burst")
    assert r0["peak"] == 3200.0 and "no probe" in r0["peak_source"]
    assert r["traffic"] >= c.frame_bytes and r["traffic_added_frame"] > r["traffic"] and "profiles/" in r["traffic_source"]


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_bench_added_frame_launches_stay_inside_the_int32_guard(name):
    """Resident.timed_added enqueues 1 + 2 n frames into one integration: never more samples than xcorr_process accepts."""
    b = _bench()
    c = wl.CONFIGS[name]
    for want in (24, 200, 10 ** 6):
        n = b.added_frames_fit(c, want)
        assert 4 <= n <= want and (2 * n + 1) * c.n_time <= 16777215


def test_bench_kstats():
    b = _bench()
    s = b.kstats([3.0, 1.0, 2.0, 10.0])
    assert s == {"mean": 4.0, "median": 2.5, "min": 1.0, "launches": 4}
