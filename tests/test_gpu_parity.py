"""GPU parity: the CUDA path (through the C ABI via the thin binding) against the CPU oracle, bit for bit.

Integer work -> the bar is exact equality (np.array_equal), no tolerance.  Small and medium shapes are compared
element by element against oracle.planar / oracle.naive on the same seeded bytes -- including shapes whose work
schedule gives every worker several segments (asserted), run as one frame, as three accumulated frames and with
xcorr_promise_complete_frames.  BASELINE.json's full-size configs are checked (a) element by element against
oracle.planar on whole channels (all 64 of C2; channels from both the data-parallel and the water-filled part of the
schedule for C4, C5, C3), (b) on sampled pairs computed one by one by oracle.pairs, (c) by the O(N*T) exact identities
of oracle/ (total power, Freivalds probes), and, as an extra, (d) whole-matrix against the standalone SIMT second opinion
of tests/support (which shares no code with libxcorr.so).
"""
import numpy as np
import pytest

import oracle
import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def xb():
    import paper_1503_06189_b200 as m
    assert torch.cuda.is_available()
    m.lib()  # must load the in-tree CUDA library; there is no fallback
    return m


def n_workers():
    return torch.cuda.get_device_properties(0).multi_processor_count // 2


def segments_per_worker(xb, n, f, t):
    """(max, min) number of work segments any worker gets in the launch configuration of this GPU."""
    _, wb = xb.xcorr_debug_schedule(n, f, t, n_workers())
    per = np.diff(wb)
    return int(per.max()), int(per.min())


def run_simt(frame):
    """The standalone SIMT second opinion (tests/support/simt_xcorr.cu) on one frame -> int32 [F][P][2]."""
    from tests import support
    out = support.simt_xcorr(torch.from_numpy(frame).cuda())
    torch.cuda.synchronize()
    return out.cpu().numpy()


def run_gpu(xb, frames, host_out=False, promise=False):
    """process every frame in `frames` (list of uint8 [T][F][N] numpy arrays), then read."""
    t, f, n = frames[0].shape
    x = xb.XCorr(n, f, t)
    if promise:
        x.promise_complete_frames()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        for fr in frames:
            d = torch.from_numpy(fr).cuda()
            x.process(d, st)
        if host_out:
            out = torch.empty((f, x.n_pairs, 2), dtype=torch.int32).pin_memory()
            x.read(out, st)
            res = out.numpy().copy()
        else:
            res = x.read(None, st)
            st.synchronize()
            res = res.cpu().numpy()
    st.synchronize()
    x.close()
    return res


# ------------------------------------------------------------------ C1 and element-by-element shapes
def test_c1_tiny_correctness_exact(xb):
    c = wl.CONFIGS["C1"]
    fr = c.frame()
    want = oracle.naive(fr)
    got = run_gpu(xb, [fr])
    assert got.shape == (4, 136, 2) and got.dtype == np.int32
    assert np.array_equal(got, want)
    assert np.array_equal(run_gpu(xb, [fr], host_out=True), want)


EDGE_SHAPES = [
    # (N, F, T, kind)  -- several tiles plus ragged tails in N (mod 128, mod 256), T (mod 32, mod 64) and odd F
    (16, 1, 1, "uniform"), (16, 3, 31, "uniform"), (48, 3, 33, "uniform"), (144, 3, 100, "uniform"),
    (208, 1, 1000, "gaussian"), (256, 5, 320, "gaussian"), (272, 2, 65, "uniform"), (400, 2, 200, "uniform"),
    (512, 3, 257, "stress"), (640, 1, 130, "gaussian_sky"), (1024, 1, 96, "uniform"),
]


@pytest.mark.parametrize("n,f,t,kind", EDGE_SHAPES)
def test_edge_shapes_exact(xb, n, f, t, kind):
    fr = wl.make_frame(kind, n, f, t, seed=n + 7 * f + t)
    assert np.array_equal(run_gpu(xb, [fr]), oracle.planar(fr))


# The symmetric block G[0:128, 128:256] of a diagonal super-tile is written half by each CTA of the pair, CTA 1's half turned
# around in registers (xengine_kernel.cuh, epilogue): input counts around the split column 192 and the block edges, so that
# CTA 1 has none, part or all of its rows 192..255 -- as one frame (plain stores) and as two added frames (staging buffer +
# bulk reduce-add), on one-tile shapes and with a ragged last diagonal tile behind an off-diagonal one.
@pytest.mark.parametrize("n", [176, 192, 208, 224, 240, 256, 448, 480, 512])
@pytest.mark.parametrize("frames", [1, 2])
def test_shared_symmetric_block_at_ragged_input_counts(xb, n, frames):
    f, t = 3, 200
    frs = [wl.make_frame("uniform" if k == 0 else "gaussian", n, f, t, seed=5 * n + k) for k in range(frames)]
    want = sum(oracle.planar(fr).astype(np.int64) for fr in frs)
    assert np.array_equal(run_gpu(xb, frs), want)


# Shapes whose schedule (xcorr_debug_schedule at this GPU's worker count) gives EVERY worker several segments, so the
# accumulator hand-off between segments (TMEM full/empty phases), the TMA prologue crossing a segment boundary, the
# water-filled split of an item along time and, for N > 256, diagonal <-> off-diagonal transitions inside one worker are
# all exercised -- and compared whole-output, element by element, with the oracle.
MULTI_SEGMENT_SHAPES = [
    # (N, F, T, kind, min segments per worker expected on 74 workers)
    (256, 160, 192, "gaussian", 2), (256, 300, 100, "uniform", 4), (256, 200, 640, "gaussian", 2),
    (512, 60, 192, "gaussian_sky", 2), (768, 40, 130, "uniform", 3), (1024, 12, 200, "stress", 1),
]


@pytest.mark.parametrize("mode", ["single", "accumulate3", "promise"])
@pytest.mark.parametrize("n,f,t,kind,min_seg", MULTI_SEGMENT_SHAPES)
def test_multi_segment_schedules_exact(xb, n, f, t, kind, min_seg, mode):
    smax, smin = segments_per_worker(xb, n, f, t)
    if n_workers() == 74:
        assert smax >= 3 and smin >= min_seg, (smax, smin)
    if mode == "single":
        fr = wl.make_frame(kind, n, f, t, seed=11 * n + f + t)
        assert np.array_equal(run_gpu(xb, [fr]), oracle.planar(fr))
        return
    frames = [wl.make_frame(kind, n, f, t, seed=11 * n + f + t + 1000 * (k + 1)) for k in range(3)]
    want = sum(oracle.planar(fr).astype(np.int64) for fr in frames)
    if mode == "accumulate3":       # frames 2 and 3 take the cp.reduce.async.bulk path into slots written by frame 1
        assert np.array_equal(run_gpu(xb, frames), want)
        return
    # promise: the first loads of a frame overlap the tail of the previous kernel of the stream; two integrations queued
    dev = [torch.from_numpy(fr).cuda() for fr in frames]
    x = xb.XCorr(n, f, t)
    x.promise_complete_frames()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        for d in dev:
            x.process(d, st)
        first = x.read(None, st)
        x.process(dev[1], st)
        second = x.read(None, st)
    torch.cuda.synchronize()
    assert np.array_equal(first.cpu().numpy(), want)
    assert np.array_equal(second.cpu().numpy(), oracle.planar(frames[1]))
    x.close()


def test_all_minus_eight_and_extremes(xb):
    # -8 is a legal value (BASELINE.json:configs[0]); every pair must be exactly 128*T
    t = 4096
    fr = wl.constant_frame(256, 2, t, 0x88)
    got = run_gpu(xb, [fr])
    assert (got[:, :, 0] == 128 * t).all() and (got[:, :, 1] == 0).all()
    # +7/-8 alternation across inputs exercises both sign corners of the int8 planes
    fr = np.empty((300, 1, 512), np.uint8)
    fr[:, :, 0::2] = 0x78   # 7 - 8i
    fr[:, :, 1::2] = 0x87   # -8 + 7i
    assert np.array_equal(run_gpu(xb, [fr]), oracle.planar(fr))


def test_zero_frame_and_one_hot(xb):
    z = np.zeros((128, 2, 256), np.uint8)
    assert not run_gpu(xb, [z]).any()
    fr = z.copy()
    fr[:, 1, 200] = wl.pack(3, -2)
    got = run_gpu(xb, [fr])
    nz = np.argwhere(got != 0)
    assert nz.tolist() == [[1, oracle.pair_index(256, 200, 200), 0]]
    assert got[1, oracle.pair_index(256, 200, 200), 0] == 128 * 13


# ------------------------------------------------------------------ accumulate / read semantics
def test_accumulates_across_process_calls_and_read_clears(xb):
    n, f, t = 256, 3, 192
    frames = [wl.gaussian_frame(n, f, t, seed=50 + k) for k in range(3)]
    want = sum(oracle.planar(fr).astype(np.int64) for fr in frames)
    both = oracle.planar(np.concatenate(frames, axis=0)).astype(np.int64)
    assert np.array_equal(want, both)                      # linearity of the oracle itself
    x = xb.XCorr(n, f, t)
    for fr in frames:
        x.process(torch.from_numpy(fr).cuda())
    got = x.read().cpu().numpy()
    assert np.array_equal(got, want)
    again = x.read().cpu().numpy()                          # second read: integration was cleared
    assert not again.any()
    x.process(torch.from_numpy(frames[1]).cuda())           # and a fresh integration starts from zero
    assert np.array_equal(x.read().cpu().numpy(), oracle.planar(frames[1]))
    assert x.kernel_launches == 3 + 1 + 1 + 1 + 1
    x.close()


def test_promise_complete_frames_is_exact(xb):
    """xcorr_promise_complete_frames: frames are loaded while the previous kernel of the stream drains; same bits.  Covers a
    read followed at once by the next integration, frames added back to back, and a frame written by torch kernels just before."""
    n, f, t = 256, 6, 700
    frames = [wl.uniform_frame(n, f, t, seed=900 + k) for k in range(4)]
    dev = [torch.from_numpy(fr).cuda() for fr in frames]
    x = xb.XCorr(n, f, t)
    x.promise_complete_frames()
    st = torch.cuda.Stream()
    outs = [torch.empty((f, x.n_pairs, 2), dtype=torch.int32, device="cuda") for _ in range(3)]
    with torch.cuda.stream(st):
        for rep in range(3):                       # process, process, read -- three integrations queued without any host sync
            x.process(dev[rep], st)
            x.process(dev[rep + 1], st)
            x.read(outs[rep], st)
        # a frame produced on the same stream immediately before xcorr_process (ordinary kernels: qualifies for the promise)
        made = (dev[0] ^ dev[3]).contiguous()
        x.process(made, st)
        last = x.read(None, st)
    torch.cuda.synchronize()
    for rep in range(3):
        want = oracle.planar(frames[rep]).astype(np.int64) + oracle.planar(frames[rep + 1])
        assert np.array_equal(outs[rep].cpu().numpy(), want)
    assert np.array_equal(last.cpu().numpy(), oracle.planar(frames[0] ^ frames[3]))
    x.promise_complete_frames(False)
    x.process(dev[2]); assert np.array_equal(x.read().cpu().numpy(), oracle.planar(frames[2]))
    x.close()


def test_error_codes_on_device(xb):
    x = xb.XCorr(16, 1, 64)
    buf = torch.zeros(16 * 64 + 16, dtype=torch.uint8, device="cuda")
    assert xb.xcorr_process(x.handle, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_process(x.handle, buf.data_ptr() + 1, 0) == xb.XCORR_EINVAL        # misaligned
    assert xb.xcorr_read(x.handle, 0, 0) == xb.XCORR_EINVAL
    with pytest.raises(ValueError):
        x.process(buf)                                                                  # wrong size
    x.close()
    # overflow guard: 128 * samples must stay below 2^31 -> at most 16,777,215 samples per integration
    x = xb.XCorr(16, 1, 8_000_000)
    big = torch.zeros(16 * 8_000_000, dtype=torch.uint8, device="cuda")
    assert xb.xcorr_process(x.handle, big.data_ptr(), 0) == xb.XCORR_OK
    assert xb.xcorr_process(x.handle, big.data_ptr(), 0) == xb.XCORR_OK
    assert xb.xcorr_process(x.handle, big.data_ptr(), 0) == xb.XCORR_EOVERFLOW
    x.read()
    assert xb.xcorr_process(x.handle, big.data_ptr(), 0) == xb.XCORR_OK
    torch.cuda.synchronize()
    x.close()


def test_int32_stays_exact_at_the_bound(xb):
    # 16,777,215 samples of -8-8i: every sum is 128 * 16,777,215 = 2^31 - 128, the largest legal value
    t = 16_777_215
    x = xb.XCorr(16, 1, t)
    fr = torch.full((t * 16,), 0x88, dtype=torch.uint8, device="cuda")
    x.process(fr)
    got = x.read().cpu().numpy()
    assert (got[:, :, 0] == 128 * t).all() and (got[:, :, 1] == 0).all()
    x.close()


def test_offset_operands_wrap_modulo_2_32(xb):
    # The tensor core is fed x + 8; the offset sums R', Q' reach 450 * T and wrap modulo 2^32 long before
    # the true visibilities (|V| <= 128 * T) leave int32.  xcorr_read's offset removal must still be exact.
    t = 16_777_215
    x = xb.XCorr(16, 1, t)
    fr = torch.empty((t, 16), dtype=torch.uint8, device="cuda")
    fr[:, 0::2] = 0x77        #  7 + 7i  -> offset operands 15, 15 (largest products)
    fr[:, 1::2] = 0x87        # -8 + 7i
    x.process(fr.reshape(-1))
    got = x.read().cpu().numpy()[0].astype(np.int64)
    x.close()
    vals = {0: 7 + 7j, 1: -8 + 7j}
    for i in range(16):
        for j in range(i, 16):
            v = vals[i % 2] * np.conj(vals[j % 2]) * t
            assert got[oracle.pair_index(16, i, j)].tolist() == [int(v.real), int(v.imag)], (i, j)


# ------------------------------------------------------------------ streamed path (a5)
def test_streamed_path_matches_oracle(xb):
    n, f, t = 256, 4, 256
    frames = [wl.gaussian_frame(n, f, t, seed=3000 + k) for k in range(5)]
    want = sum(oracle.planar(fr).astype(np.int64) for fr in frames)
    x = xb.XCorr(n, f, t)
    s = xb.XCorrStream(x, depth=2)
    pinned = [torch.from_numpy(fr).pin_memory() for fr in frames]
    for p in pinned:
        s.submit(p)
    out = torch.empty((f, x.n_pairs, 2), dtype=torch.int32).pin_memory()
    s.read(out)
    assert np.array_equal(out.numpy(), want)
    # pageable host memory and a device output also work
    for fr in frames[:2]:
        s.submit(fr)
    dout = torch.empty((f, x.n_pairs, 2), dtype=torch.int32, device="cuda")
    s.read(dout)
    assert np.array_equal(dout.cpu().numpy(), oracle.planar(frames[0]).astype(np.int64) + oracle.planar(frames[1]))
    # asynchronous reads: one integration per frame, the next submit follows at once, results valid after sync()
    outs = [torch.empty((f, x.n_pairs, 2), dtype=torch.int32).pin_memory() for _ in frames]
    for p, o in zip(pinned, outs):
        s.submit(p)
        s.read_async(o)
    s.sync()
    for fr, o in zip(frames, outs):
        assert np.array_equal(o.numpy(), oracle.planar(fr))
    s.close()
    x.close()


# ------------------------------------------------------------------ full-size configs
def _sample_pairs(rng, n, f, k, extra=()):
    i = rng.integers(0, n, size=k)
    j = rng.integers(0, n, size=k)
    lo, hi = np.minimum(i, j), np.maximum(i, j)
    ch = rng.integers(0, f, size=k)
    idx = np.stack([ch, lo, hi], axis=1).astype(np.int32)
    if len(extra):
        idx = np.concatenate([idx, np.asarray(extra, np.int32)])
    return idx


def _check_full_size(fr, got, n_samples=1500, n_probe=2, channels=None, seed=0):
    """Sampled exact pairs + exact O(N*T) identities for a [F][P][2] result on frame fr."""
    t, f, n = fr.shape
    rng = np.random.default_rng(seed)
    assert n >= 256
    corners = [(0, 0, 0), (f - 1, n - 1, n - 1), (0, 0, n - 1), (f - 1, 127, 128), (0, 255, 255), (f // 2, 128, 128)]
    if n > 256:
        corners += [(0, 255, 256), (f - 1, 0, 256), (0, 256, n - 1), (0, 300, 300)]
    idx = _sample_pairs(rng, n, f, n_samples, corners)
    want = oracle.pairs(fr, idx)
    p = idx[:, 1].astype(np.int64) * (2 * n - idx[:, 1] + 1) // 2 + (idx[:, 2] - idx[:, 1])
    assert np.array_equal(got[idx[:, 0], p].astype(np.int64), want)
    chans = range(f) if channels is None else channels
    tp = None
    for ch in chans:
        fch = np.ascontiguousarray(fr[:, ch, :])
        tri = got[ch]
        # identity 1: sum_i V_ii + 2 sum_{i<j} Re V_ij == sum_t |sum_n x_n|^2
        assert oracle.lhs_total_power(tri[None], n)[0] == oracle.identity_total_power(fch[:, None, :])[0]
        for _ in range(n_probe):
            u = rng.integers(-2, 3, size=n)
            w = rng.integers(-2, 3, size=n)
            assert oracle.freivalds_lhs(tri, n, u, w) == oracle.freivalds_rhs(fch, u, w)


def _channels(fr, chans):
    """oracle.planar on the listed whole channels of a frame -> int32 [len(chans)][P][2]."""
    return oracle.planar(np.ascontiguousarray(fr[:, list(chans), :]))


def test_c2_full_size(xb):
    c = wl.CONFIGS["C2"]
    fr = c.frame()
    assert fr.nbytes == 268_435_456
    smax, _ = segments_per_worker(xb, c.n_inputs, c.n_freq, c.n_time)
    assert smax >= 2                      # every item is cut in time between two workers (64 items on 74 workers)
    got = run_gpu(xb, [fr])
    assert got.nbytes == 16_842_752
    # whole output, all 64 channels, every element, against the oracle
    assert np.array_equal(got, oracle.planar(fr))
    _check_full_size(fr, got, channels=range(0, 64, 7))
    # the same with the promise bench.py runs under
    assert np.array_equal(run_gpu(xb, [fr], promise=True), got)
    # extra: the standalone SIMT second opinion agrees as well
    assert np.array_equal(got, run_simt(fr))


def test_c4_full_size(xb):
    c = wl.CONFIGS["C4"]
    fr = c.frame()
    got = run_gpu(xb, [fr])
    # whole channels against the oracle: 0 and 7 from the data-parallel part of the schedule (items that run whole on one
    # worker), 14 and 15 from the water-filled remainder (items cut in time, up to 9 segments per worker)
    seg, wb = xb.xcorr_debug_schedule(c.n_inputs, c.n_freq, c.n_time, n_workers())
    n_stage = -(-c.n_time // xb.xcorr_debug_stage_samples())
    whole = {int(s[0]) for s in seg if s[4] - s[3] == n_stage}
    cut = {int(s[0]) for s in seg if s[4] - s[3] < n_stage}
    chans = [0, 7, 14, 15]
    assert {0, 7} <= whole and {14, 15} & cut
    assert np.array_equal(got[chans], _channels(fr, chans))
    _check_full_size(fr, got, n_samples=3000, channels=[3, 11])
    assert np.array_equal(got, run_simt(fr))             # extra: whole matrix against the SIMT second opinion
    # the common sky signal makes off-diagonal real parts positive on average (~2*T)
    off = got[0, 1:2048, 0].astype(np.float64)
    assert 1.0 < off.mean() / c.n_time < 3.0


def test_c5_full_size_stress(xb):
    c = wl.CONFIGS["C5"]
    fr = c.frame()
    assert fr.nbytes == 2 ** 31
    got = run_gpu(xb, [fr])
    n, t = c.n_inputs, c.n_time
    # const-const pairs (inputs < 256): exactly (128*T, 0) = (16,777,216, 0)
    for i in (0, 1, 127, 128, 255):
        for j in (i, 255):
            assert got[:, oracle.pair_index(n, i, j)].tolist() == [[128 * t, 0]] * c.n_freq
    blk = np.concatenate([np.arange(oracle.pair_index(n, i, i), oracle.pair_index(n, i, 255) + 1) for i in range(256)])
    assert (got[:, blk, 0] == 128 * t).all() and (got[:, blk, 1] == 0).all()
    # const-random pairs: V[i,j] = (-8-8i) * conj(sum_t x_j)
    re, im = oracle.unpack(fr[:, 3, 256:])
    sr, si = re.sum(0), im.sum(0)
    for i in (0, 200):
        seg = got[3, oracle.pair_index(n, i, 256): oracle.pair_index(n, i, 511) + 1]
        assert np.array_equal(seg[:, 0], -8 * sr - 8 * si) and np.array_equal(seg[:, 1], 8 * si - 8 * sr)
    # whole channels against the oracle: 0 (data-parallel part of the schedule), 24 and 31 (water-filled remainder)
    chans = [0, 24, 31]
    assert np.array_equal(got[chans], _channels(fr, chans))
    _check_full_size(fr, got, n_samples=1200, channels=[12], n_probe=1)
    assert np.array_equal(got, run_simt(fr))             # extra
    # steady state of long segments (2048 stages per item), many launches back to back with the promise on: the two unpack
    # groups of a CTA drift apart and TMA loads land out of order -- a packed slot consumed by alternating groups once let a
    # group pass its full-barrier wait on a stale phase parity here (xengine_kernel.cuh, kPackedStages % kUnpackGroups).
    # Every launch must reproduce the result verified above.
    x = xb.XCorr(c.n_inputs, c.n_freq, c.n_time)
    x.promise_complete_frames()
    dev = torch.from_numpy(fr).cuda()
    st = torch.cuda.Stream()
    outs = [torch.empty((c.n_freq, x.n_pairs, 2), dtype=torch.int32, device="cuda") for _ in range(12)]
    with torch.cuda.stream(st):
        for o in outs:
            x.process(dev, st)
            x.read(o, st)
    torch.cuda.synchronize()
    want = torch.from_numpy(got).cuda()
    for k, o in enumerate(outs):
        assert torch.equal(o, want), k
    x.close()


def test_c4_two_distinct_frames_added_full_size(xb):
    """The telescope's steady state at full size (the kernels "simply add to the output of the last run"): two
    distinct C4 frames into one integration -- the second takes the added-frame epilogue (bulk reduce-adds) on every tile of
    the N = 2048 schedule -- against the sum of the oracle's results: whole channels from both schedule regimes, sampled
    pairs over all channels, the total-power identity on two more channels."""
    c = wl.CONFIGS["C4"]
    frames = [c.frame(0), c.frame(1)]
    assert not np.array_equal(frames[0][:64], frames[1][:64])
    got = run_gpu(xb, frames, promise=True)
    chans = [0, 7, 14, 15]
    want = sum(_channels(fr, chans).astype(np.int64) for fr in frames)
    assert np.array_equal(got[chans], want)
    n, f = c.n_inputs, c.n_freq
    rng = np.random.default_rng(41)
    idx = _sample_pairs(rng, n, f, 3000, [(0, 0, 0), (f - 1, n - 1, n - 1), (0, 255, 256), (f - 1, 0, n - 1), (5, 1023, 1024)])
    p = idx[:, 1].astype(np.int64) * (2 * n - idx[:, 1] + 1) // 2 + (idx[:, 2] - idx[:, 1])
    assert np.array_equal(got[idx[:, 0], p].astype(np.int64), sum(oracle.pairs(fr, idx).astype(np.int64) for fr in frames))
    for ch in (3, 11):
        tp = sum(int(oracle.identity_total_power(np.ascontiguousarray(fr[:, ch, :])[:, None, :])[0]) for fr in frames)
        assert int(oracle.lhs_total_power(got[ch][None], n)[0]) == tp


def test_c5_frame_processed_twice_full_size(xb):
    """C5 (2 GiB frame, 2048 stages per item) processed TWICE into one integration: first-frame epilogue, then the added-frame
    epilogue on every tile; by linearity the result is exactly 2 x the oracle's -- whole channels from both schedule regimes,
    the closed form of the constant block on all channels, sampled pairs elsewhere."""
    c = wl.CONFIGS["C5"]
    fr = c.frame()
    got = run_gpu(xb, [fr, fr], promise=True)
    n, f, t = c.n_inputs, c.n_freq, c.n_time
    chans = [0, 24, 31]
    assert np.array_equal(got[chans], 2 * _channels(fr, chans).astype(np.int64))
    blk = np.concatenate([np.arange(oracle.pair_index(n, i, i), oracle.pair_index(n, i, 255) + 1) for i in range(256)])
    assert (got[:, blk, 0] == 2 * 128 * t).all() and (got[:, blk, 1] == 0).all()
    rng = np.random.default_rng(43)
    idx = _sample_pairs(rng, n, f, 1200, [(0, 255, 256), (f - 1, 0, 511), (7, 300, 300), (f - 1, 511, 511)])
    p = idx[:, 1].astype(np.int64) * (2 * n - idx[:, 1] + 1) // 2 + (idx[:, 2] - idx[:, 1])
    assert np.array_equal(got[idx[:, 0], p].astype(np.int64), 2 * oracle.pairs(fr, idx).astype(np.int64))


C3_POOL = 4   # distinct seeded 1 GiB frames, cycled 16 times = the 64 consecutive frames of BASELINE.json:configs[2]


def test_c3_streamed_64_frames(xb):
    """C3 as specified: N=256, F=1024, T=4096 (1 GiB frames), 64 frames streamed from pinned host memory through the
    double-buffered H2D ring with the promise bench.py uses, ONE read at the end.  The 64 frames are a pool of C3_POOL = 4
    distinct seeded frames cycled 16 times; by linearity the result must be 16 * sum_p oracle(frame_p)."""
    c = wl.CONFIGS["C3"]
    assert c.n_frames == 64 and 64 % C3_POOL == 0
    reps = c.n_frames // C3_POOL
    pool = [torch.from_numpy(c.frame(k)).pin_memory() for k in range(C3_POOL)]
    smax, smin = segments_per_worker(xb, c.n_inputs, c.n_freq, c.n_time)
    assert smax >= 3 and smin >= 3
    x = xb.XCorr(c.n_inputs, c.n_freq, c.n_time)
    x.promise_complete_frames()
    s = xb.XCorrStream(x, depth=2)
    for k in range(c.n_frames):
        s.submit(pool[k % C3_POOL])
    out = torch.empty((c.n_freq, x.n_pairs, 2), dtype=torch.int32).pin_memory()
    s.read(out)
    got = out.numpy()
    s.close()
    x.close()
    # whole channels, element by element: first, last, and some in between (every worker's segment list is touched)
    chans = [0, 1, 73, 74, 511, 1000, 1023]
    want = sum(_channels(p.numpy(), chans).astype(np.int64) for p in pool) * reps
    assert np.array_equal(got[chans], want)
    rng = np.random.default_rng(5)
    idx = _sample_pairs(rng, 256, 1024, 1500)
    want = reps * sum(oracle.pairs(p.numpy(), idx) for p in pool)
    pp = idx[:, 1].astype(np.int64) * (2 * 256 - idx[:, 1] + 1) // 2 + (idx[:, 2] - idx[:, 1])
    assert np.array_equal(got[idx[:, 0], pp].astype(np.int64), want)
    # total-power identity on every 16th channel (linear in the frame, so it sums over the 64 frames too)
    for ch in range(0, 1024, 16):
        rhs = reps * sum(int(oracle.identity_total_power(np.ascontiguousarray(p.numpy()[:, ch:ch + 1, :]))[0]) for p in pool)
        assert int(oracle.lhs_total_power(got[ch:ch + 1], 256)[0]) == rhs
    # extra: the whole 269 MB result against the SIMT second opinion, frame by frame
    ref = sum(run_simt(p.numpy()).astype(np.int64) for p in pool) * reps
    assert np.array_equal(got, ref)


# ------------------------------------------------------------------ streamed path with the promise (bench.py's e2e configuration)
def test_streamed_path_with_promise_distinct_frames_per_slot(xb):
    """xcorr_stream_submit + read_async, depth 2, promise on, 7 distinct frames (so each ring slot is rewritten with new
    data several times while the previous kernel may still be draining) -- shapes with several segments per worker."""
    for (n, f, t) in [(256, 160, 192), (512, 60, 192)]:
        frames = [wl.gaussian_frame(n, f, t, seed=7000 + n + k) for k in range(7)]
        pinned = [torch.from_numpy(fr).pin_memory() for fr in frames]
        x = xb.XCorr(n, f, t)
        x.promise_complete_frames()
        s = xb.XCorrStream(x, depth=2)
        outs = [torch.empty((f, x.n_pairs, 2), dtype=torch.int32).pin_memory() for _ in frames]
        for p_, o in zip(pinned, outs):          # one integration per frame, nothing waits in between
            s.submit(p_)
            s.read_async(o)
        s.sync()
        for fr, o in zip(frames, outs):
            assert np.array_equal(o.numpy(), oracle.planar(fr))
        for p_ in pinned:                        # and all seven into one integration
            s.submit(p_)
        out = torch.empty((f, x.n_pairs, 2), dtype=torch.int32).pin_memory()
        s.read(out)
        assert np.array_equal(out.numpy(), sum(oracle.planar(fr).astype(np.int64) for fr in frames))
        s.close()
        x.close()


# ------------------------------------------------------------------ handle state across streams
def test_process_and_read_on_different_streams_are_ordered(xb):
    """include/xcorr.h: a call on another stream than the handle's previous call waits, on the device, for that call's work."""
    n, f, t = 256, 160, 192
    frames = [wl.uniform_frame(n, f, t, seed=8100 + k) for k in range(3)]
    dev = [torch.from_numpy(fr).cuda() for fr in frames]
    torch.cuda.synchronize()
    x = xb.XCorr(n, f, t)
    sa, sb, sc = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for rep in range(4):
        x.process(dev[0], sa)
        x.process(dev[1], sb)        # another stream: must see frame 0's slots
        outs.append(x.read(None, sc))  # a third one: must see both
        x.process(dev[2], sa)        # next integration, back on the first stream: must not overtake the read
        outs.append(x.read(None, sb))
    torch.cuda.synchronize()
    want01 = oracle.planar(frames[0]).astype(np.int64) + oracle.planar(frames[1])
    want2 = oracle.planar(frames[2])
    for k, o in enumerate(outs):
        assert np.array_equal(o.cpu().numpy(), want01 if k % 2 == 0 else want2), k
    x.close()


def test_wrapper_keeps_a_temporary_stream_alive_until_the_next_call(xb):
    """include/xcorr.h: the stream of a call must outlive the handle's next call (that call records an event on it).  A
    torch stream created for one ``process`` and dropped at once would break that; ``XCorr`` keeps the object referenced."""
    import gc
    n, f, t = 64, 16, 256
    frames = [wl.uniform_frame(n, f, t, seed=8200 + k) for k in range(2)]
    dev = [torch.from_numpy(fr).cuda() for fr in frames]
    torch.cuda.synchronize()
    x = xb.XCorr(n, f, t)
    keep = torch.cuda.Stream()
    for rep in range(3):
        x.process(dev[0], torch.cuda.Stream())     # temporary: no other reference than the wrapper's
        gc.collect()
        assert isinstance(x._last_stream, torch.cuda.Stream)
        x.process(dev[1], torch.cuda.Stream())
        gc.collect()
        got = x.read(None, keep)
        torch.cuda.synchronize()
        assert np.array_equal(got.cpu().numpy(), oracle.planar(frames[0]).astype(np.int64) + oracle.planar(frames[1]))
    x.close()


# ------------------------------------------------------------------ modulo-2^32 behaviour of the offset sums inside a slot
def test_offset_sums_wrap_inside_tmem_and_inside_a_slot(xb):
    """The tensor core is fed offset operands, so the sums held in TMEM and in an accumulator slot grow far
    faster than the visibilities (up to 900 per sample against 128) and wrap modulo 2^32 long before the int32 guard
    (16,777,215 samples).  F = n_workers channels of N = 16: every item runs whole on one worker, so ONE TMEM accumulator
    integrates all T = 5,000,000 samples of a frame (wraps in TMEM), and three frames are reduce-added into the same slot
    (wraps in cp.reduce.async.bulk .add.s32).  Closed form per pair."""
    w = n_workers()
    n, f, t = 16, w, 5_000_000
    seg, wb = xb.xcorr_debug_schedule(n, f, t, w)
    assert len(seg) == f and (np.diff(wb) == 1).all()            # one whole item per worker
    fr = torch.empty((t, f, n), dtype=torch.uint8, device="cuda")
    fr[:, :, 0::2] = 0x77        #  7 + 7i  -> offset operands 15, 15 (largest products)
    fr[:, :, 1::2] = 0x87        # -8 + 7i
    x = xb.XCorr(n, f, t)
    for _ in range(3):
        x.process(fr.reshape(-1))
    got = x.read().cpu().numpy().astype(np.int64)
    x.close()
    vals = {0: 7 + 7j, 1: -8 + 7j}
    want = np.zeros((n * (n + 1) // 2, 2), dtype=np.int64)
    for i in range(n):
        for j in range(i, n):
            v = vals[i % 2] * np.conj(vals[j % 2]) * (3 * t)
            want[oracle.pair_index(n, i, j)] = (int(v.real), int(v.imag))
    assert np.array_equal(got, np.broadcast_to(want, got.shape))


# ------------------------------------------------------------------ NEXT-3: several handles on disjoint channel ranges
@pytest.mark.parametrize("split", ["two_ranks", "streams_3_3_2"])
def test_channel_range_replicas_through_the_c_abi(xb, split):
    """Each GPU of a server correlates its own streams' channels; the merged result is the concatenation along f
    (PAPER.md:51 "each of the AMD R9 280X GPUs processes 3 of these streams, and the R9 270X processes 2"; :111 "combines
    all eight streams").  Here: one handle per channel range on one GPU, each fed its slice of the frame."""
    from paper_1503_06189_b200 import replicas
    n, f, t = 256, 64, 320
    if split == "two_ranks":
        ranges = replicas.channel_ranges(f, 2)
    else:
        ranges, b = [], 0
        for n_streams in (3, 3, 2):                          # 8 streams of 8 channels
            ranges.append((b, b + 8 * n_streams))
            b += 8 * n_streams
        assert b == f
    frames = [wl.gaussian_frame(n, f, t, seed=8200 + k) for k in range(2)]
    handles = [xb.XCorr(n, e - b, t) for b, e in ranges]
    streams = [torch.cuda.Stream() for _ in ranges]
    for fr in frames:
        for (b, e), x, st in zip(ranges, handles, streams):
            with torch.cuda.stream(st):
                x.process(torch.from_numpy(np.ascontiguousarray(fr[:, b:e, :])).cuda(), st)
    parts = [x.read(None, st) for x, st in zip(handles, streams)]
    torch.cuda.synchronize()
    merged = np.concatenate([p.cpu().numpy() for p in parts], axis=0)
    want = sum(oracle.planar(fr).astype(np.int64) for fr in frames)
    assert np.array_equal(merged, want)
    for x in handles:
        x.close()
