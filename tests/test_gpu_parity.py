"""GPU parity: the CUDA path (through the C ABI via the thin binding) against the CPU oracle, bit for bit.

Integer work -> the bar is exact equality (np.array_equal), no tolerance.  Small and medium shapes are compared
element by element against oracle.planar / oracle.naive on the same seeded bytes; BASELINE.json's full-size
configs are checked (a) on sampled pairs computed one by one by oracle.pairs, (b) by the O(N*T) exact identities
of oracle/ (total power, Freivalds probes) over every channel, and (c) whole-matrix against the on-device SIMT
second opinion, which is itself held to (a) and (b).
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


def run_gpu(xb, frames, simt=False, host_out=False):
    """process every frame in `frames` (list of uint8 [T][F][N] numpy arrays), then read."""
    t, f, n = frames[0].shape
    x = xb.XCorr(n, f, t)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        for fr in frames:
            d = torch.from_numpy(fr).cuda()
            (x.process_simt_debug if simt else x.process)(d, st)
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


def test_c2_full_size(xb):
    c = wl.CONFIGS["C2"]
    fr = c.frame()
    assert fr.nbytes == 268_435_456
    got = run_gpu(xb, [fr])
    assert got.nbytes == 16_842_752
    _check_full_size(fr, got, channels=range(0, 64, 3))
    # whole matrix, every element: against the SIMT second opinion (held to the same oracle checks above)
    ref = run_gpu(xb, [fr], simt=True)
    assert np.array_equal(got, ref)
    # two channels in full against the oracle
    part = oracle.planar(fr, 17, 19)
    assert np.array_equal(got[17:19], part[17:19])


def test_c4_full_size(xb):
    c = wl.CONFIGS["C4"]
    fr = c.frame()
    got = run_gpu(xb, [fr])
    _check_full_size(fr, got, n_samples=3000, channels=[0, 7, 15])
    ref = run_gpu(xb, [fr], simt=True)
    assert np.array_equal(got, ref)
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
    _check_full_size(fr, got, n_samples=1200, channels=[0, 31], n_probe=1)
    ref = run_gpu(xb, [fr], simt=True)
    assert np.array_equal(got, ref)


def test_c3_streamed_shape_reduced_frames(xb):
    # C3's shape (N=256, F=1024, T=4096, 1 GiB frames) streamed from pinned memory; a pool of 2 distinct seeded
    # frames is cycled 3 times (6 frames) -- by linearity the result must be 3 * (oracle(A) + oracle(B)).
    c = wl.CONFIGS["C3"]
    pool = [torch.from_numpy(c.frame(k)).pin_memory() for k in range(2)]
    x = xb.XCorr(c.n_inputs, c.n_freq, c.n_time)
    s = xb.XCorrStream(x, depth=2)
    for rep in range(3):
        for p in pool:
            s.submit(p)
    out = torch.empty((c.n_freq, x.n_pairs, 2), dtype=torch.int32).pin_memory()
    s.read(out)
    got = out.numpy()
    s.close()
    x.close()
    chans = [0, 511, 1023]
    want = sum(oracle.planar(np.ascontiguousarray(p.numpy()[:, chans, :])).astype(np.int64) for p in pool) * 3
    assert np.array_equal(got[chans], want)
    rng = np.random.default_rng(5)
    idx = _sample_pairs(rng, 256, 1024, 1500)
    want = 3 * sum(oracle.pairs(p.numpy(), idx) for p in pool)
    pp = idx[:, 1].astype(np.int64) * (2 * 256 - idx[:, 1] + 1) // 2 + (idx[:, 2] - idx[:, 1])
    assert np.array_equal(got[idx[:, 0], pp].astype(np.int64), want)
    # total-power identity on every 16th channel (linear in the frame, so it sums over the 6 frames too)
    for ch in range(0, 1024, 16):
        rhs = 3 * sum(int(oracle.identity_total_power(np.ascontiguousarray(p.numpy()[:, ch:ch + 1, :]))[0]) for p in pool)
        assert int(oracle.lhs_total_power(got[ch:ch + 1], 256)[0]) == rhs
