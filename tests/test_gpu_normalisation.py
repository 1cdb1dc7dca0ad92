"""GPU parity for the lost-sample normalisation (NEXT-1): flag_count_kernel + finalize_kernel<true>
through the C ABI, against oracle/normalisation.py on the same seeded flags, loss counters and frames.

Bar: the normalisation matrix L is integer work -> bit-exact.  The normalised visibilities are float32 computed as
float(V) * (float(T) / float(T - L)) with round-to-nearest at each of the three steps (int32 -> float conversion,
division, multiplication): relative error <= 3 * 2^-24 (1 + O(2^-24)) against the float64 oracle, tested at
rtol = 2^-22; zeros (no valid sample, or V = 0) must be exact.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from oracle import normalisation as on

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

RTOL = 2.0 ** -22


@pytest.fixture(scope="module")
def xb():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1503_06189_b200 as xb
    return xb


def run(xb, n, f, t, frames, flags_list, lost_list, want_lost=True):
    x = xb.XCorr(n, f, t)
    x.norm_enable()
    for fr, fl, lo in zip(frames, flags_list, lost_list):
        x.process(torch.from_numpy(fr).cuda())
        x.norm_process(None if fl is None else torch.from_numpy(wl.pack_flags(fl)).cuda(), lo)
    lost_out = torch.empty((f, x.n_pairs), dtype=torch.int32, device="cuda") if want_lost else None
    vis = x.read_normalized(lost_out=lost_out)
    torch.cuda.synchronize()
    return x, vis.cpu().numpy(), (lost_out.cpu().numpy() if want_lost else None)


def check_vis(got, want):
    assert got.dtype == np.float32
    zero = want == 0
    assert not got[zero].any()
    assert np.allclose(got[~zero].astype(np.float64), want[~zero], rtol=RTOL, atol=0.0)


@pytest.mark.parametrize("n,f,t,dense", [(16, 4, 256, True), (48, 3, 100, True), (144, 1, 65, True), (256, 8, 512, False),
                                         (272, 2, 257, True), (512, 2, 200, False),
                                         # several work segments per worker (3 at most, 2 at least on 74 workers): the slots of a
                                         # tile are summed and normalised in one pass
                                         (256, 160, 192, False), (512, 60, 192, True)])
def test_normalisation_matches_oracle(xb, n, f, t, dense):
    if (n, f, t) in ((256, 160, 192), (512, 60, 192)):
        _, wb = xb.xcorr_debug_schedule(n, f, t, 74)
        assert np.diff(wb).max() >= 3
    kw = dict(p_flag=0.03, p_burst=0.05, burst_frac=0.2, p_packet_loss=0.08) if dense else {}
    flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, 21, **kw)
    fr = wl.zero_lost_samples(wl.make_frame("gaussian", n, f, t, 22), flags, lost_mask)
    x, vis, L = run(xb, n, f, t, [fr], [flags], [lost])
    want_l = on.lost_matrix(flags, lost)
    assert np.array_equal(L, want_l)
    check_vis(vis, on.normalise(oracle.planar(fr), t, want_l))
    x.close()


def test_accumulates_over_frames_and_read_clears(xb):
    n, f, t = 64, 8, 96
    fls, los, frs = [], [], []
    for k in range(3):
        flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, 30 + k, p_flag=0.02, p_burst=0.05, burst_frac=0.3, p_packet_loss=0.1)
        fls.append(flags); los.append(lost)
        frs.append(wl.zero_lost_samples(wl.make_frame("uniform", n, f, t, 40 + k), flags, lost_mask))
    x, vis, L = run(xb, n, f, t, frs, fls, los)
    want_l = sum(on.lost_matrix(fl, lo) for fl, lo in zip(fls, los))
    assert np.array_equal(L, want_l)
    want_v = sum(oracle.planar(fr).astype(np.int64) for fr in frs)
    check_vis(vis, on.normalise(want_v, 3 * t, want_l))
    # the read ended the integration: flags and loss counters start from zero again
    x.process(torch.from_numpy(frs[0]).cuda())
    lost_out = torch.empty((f, x.n_pairs), dtype=torch.int32, device="cuda")
    vis2 = x.read_normalized(lost_out=lost_out).cpu().numpy()
    assert not lost_out.cpu().numpy().any()
    assert np.array_equal(vis2, oracle.planar(frs[0]).astype(np.float32))
    # a plain xcorr_read ends the integration for the flag state as well
    x.process(torch.from_numpy(frs[1]).cuda())
    x.norm_process(torch.from_numpy(wl.pack_flags(fls[1])).cuda(), los[1])
    assert np.array_equal(x.read().cpu().numpy(), oracle.planar(frs[1]))
    x.process(torch.from_numpy(frs[2]).cuda())
    x.read_normalized(lost_out=lost_out)
    assert not lost_out.cpu().numpy().any()
    x.close()


def test_flags_only_loss_only_and_host_outputs(xb):
    n, f, t = 32, 3, 64
    flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, 50, p_flag=0.05, p_packet_loss=0.2)
    fr = wl.zero_lost_samples(wl.make_frame("uniform", n, f, t, 51), flags, lost_mask)
    want_l = on.lost_matrix(flags, lost)
    want_v = on.normalise(oracle.planar(fr), t, want_l)
    x = xb.XCorr(n, f, t)
    x.norm_enable()
    x.norm_enable()                                    # idempotent
    x.process(torch.from_numpy(fr).cuda())
    x.norm_process(torch.from_numpy(wl.pack_flags(flags)).cuda(), None)     # two calls: flags, then the loss counters
    x.norm_process(None, lost)
    out = torch.empty((f, x.n_pairs, 2), dtype=torch.float32)               # host outputs
    lout = torch.empty((f, x.n_pairs), dtype=torch.int32)
    x.read_normalized(out, lout)
    assert np.array_equal(lout.numpy(), want_l)
    check_vis(out.numpy(), want_v)
    x.close()


def test_all_flagged_sample_and_everything_lost(xb):
    n, f, t = 16, 2, 8
    flags = np.zeros((t, f, n), dtype=bool)
    flags[3, 0, :] = True                              # E = N: every input flagged in one sample
    lost = np.array([0, t], dtype=np.int32)            # channel 1 lost completely
    lost_mask = np.zeros((t, f), dtype=bool)
    lost_mask[:, 1] = True
    fr = wl.zero_lost_samples(wl.make_frame("uniform", n, f, t, 3), flags, lost_mask)
    x, vis, L = run(xb, n, f, t, [fr], [flags], [lost])
    assert (L[0] == 1).all() and (L[1] == t).all()
    assert not vis[1].any() and np.isfinite(vis).all()
    check_vis(vis, on.normalise(oracle.planar(fr), t, on.lost_matrix(flags, lost)))
    x.close()


def test_errors(xb):
    x = xb.XCorr(16, 1, 8)
    assert xb.xcorr_norm_process(x.handle, 0, 0, 0) == xb.XCORR_EINVAL          # not enabled
    out = torch.empty((1, x.n_pairs, 2), dtype=torch.float32, device="cuda")
    assert xb.xcorr_read_normalized(x.handle, out.data_ptr(), 0, 0) == xb.XCORR_EINVAL
    x.norm_enable()
    bad = np.array([9], dtype=np.int32)                                            # more lost samples than the frame has
    assert xb.xcorr_norm_process(x.handle, 0, bad.ctypes.data, 0) == xb.XCORR_EINVAL
    fl = torch.zeros(32, dtype=torch.uint8, device="cuda")
    assert xb.xcorr_norm_process(x.handle, fl.data_ptr() + 1, 0, 0) == xb.XCORR_EINVAL   # misaligned
    x.close()


def test_c2_full_size_normalised(xb):
    """BASELINE.json:configs[1] shape with this build's flag / loss rates."""
    c = wl.CONFIGS["C2"]
    n, f, t = c.n_inputs, c.n_freq, c.n_time
    flags, lost_mask, lost = wl.draw_flags_and_loss(n, f, t, 77)
    fr = wl.zero_lost_samples(c.frame(), flags, lost_mask)
    x, vis, L = run(xb, n, f, t, [fr], [flags], [lost])
    x.close()
    # sampled pairs, each checked from the definition: T - #{samples with both inputs present}, and V by the oracle
    rng = np.random.default_rng(9)
    k = 600
    i = rng.integers(0, n, k); j = rng.integers(0, n, k)
    lo, hi = np.minimum(i, j), np.maximum(i, j)
    ch = rng.integers(0, f, k)
    idx = np.stack([ch, lo, hi], axis=1).astype(np.int32)
    present = ~flags & ~lost_mask[:, :, None]
    p = lo.astype(np.int64) * (2 * n - lo + 1) // 2 + (hi - lo)
    valid = np.array([(present[:, c_, a] & present[:, c_, b]).sum() for c_, a, b in idx])
    assert np.array_equal(L[ch, p], t - valid)
    v = oracle.pairs(fr, idx).astype(np.float64)
    want = v * (t / valid)[:, None]
    assert np.allclose(vis[ch, p].astype(np.float64), want, rtol=RTOL, atol=0.0)
    # whole matrix of four channels against the step-by-step oracle
    for c_ in (0, 21, 42, 63):
        want_l = on.lost_matrix(flags[:, c_:c_ + 1], lost[c_:c_ + 1])
        assert np.array_equal(L[c_:c_ + 1], want_l)
        check_vis(vis[c_:c_ + 1], on.normalise(oracle.planar(np.ascontiguousarray(fr[:, c_:c_ + 1])), t, want_l))
