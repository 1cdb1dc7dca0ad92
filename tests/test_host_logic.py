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
