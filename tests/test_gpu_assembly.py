"""GPU parity of packet -> frame assembly (NEXT-2) against oracle/assembly.py: byte-exact frame, flag field, counters."""
import numpy as np
import pytest

import oracle
import oracle.assembly as oa
import oracle.normalisation as on
import workloads as wl

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def xb():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1503_06189_b200 as xb
    return xb


def make_case(n, f, t, seed, S=4, C=8, p_loss=0.03, p_dup=0.03, p_late=0.1, n_foreign=5, kind="uniform", seq0=123456789012):
    fr = wl.make_frame(kind, n, f, t, seed)
    flags, _, _ = wl.draw_flags_and_loss(n, f, t, seed + 1, p_flag=5e-3, p_burst=5e-3, burst_frac=0.1, p_packet_loss=0.0)
    pk = wl.packetise(fr, wl.pack_flags(flags), seq0, S, C)
    return wl.disturb_packets(pk, seed + 2, p_loss=p_loss, p_dup=p_dup, p_late=p_late, n_foreign=n_foreign), seq0


def run_gpu(xb, arrived, n, f, t, seq0, S=4, C=8, pinned=False):
    a = xb.Assembler(n, f, t, S, C)
    assert a.packet_bytes == oa.packet_bytes(n, S, C)
    flat = torch.from_numpy(arrived.reshape(-1))
    pk = flat.pin_memory() if pinned else flat.cuda()
    # poison the outputs: every byte must be written by the kernels (no clearing pass)
    frame = torch.full((t, f, n), 0xA5, dtype=torch.uint8, device="cuda")
    flags = torch.full((t, f, n // 8), 0xA5, dtype=torch.uint8, device="cuda")
    frame, flags, lost, counts = a.assemble(pk if arrived.shape[0] else None, arrived.shape[0], seq0, frame=frame, flags=flags)
    torch.cuda.synchronize()
    assert a.kernel_launches == 2
    out = frame.cpu().numpy(), flags.cpu().numpy(), lost.cpu().numpy(), counts.cpu().numpy()
    a.close()
    return out


def check(got, want):
    frame, flags, lost, counts = got
    assert np.array_equal(frame, want["frame"])
    assert np.array_equal(flags, want["flags"])
    assert np.array_equal(lost.astype(np.int64), want["lost"])
    assert counts[:3].tolist() == [want["kept"], want["duplicates"], want["rejected"]]


@pytest.mark.parametrize("n,f,t,S,C", [(16, 8, 16, 4, 8), (48, 16, 100, 4, 8), (256, 16, 64, 4, 8), (144, 8, 66, 2, 8), (16, 32, 24, 1, 16),
                                       (272, 24, 40, 8, 8), (1024, 8, 16, 4, 8)])
def test_assembly_matches_oracle(xb, n, f, t, S, C):
    arrived, seq0 = make_case(n, f, t, 100 + n, S, C, p_loss=0.15, p_dup=0.1, p_late=0.2)
    want = oa.assemble(arrived, n, f, t, seq0, S, C)
    assert want["rejected"] == 5
    check(run_gpu(xb, arrived, n, f, t, seq0, S, C), want)


def test_packets_in_pinned_host_memory(xb):
    n, f, t = 256, 16, 128
    arrived, seq0 = make_case(n, f, t, 7)
    check(run_gpu(xb, arrived, n, f, t, seq0, pinned=True), oa.assemble(arrived, n, f, t, seq0))


def test_first_arrival_wins_when_a_duplicate_differs(xb):
    n, f, t = 16, 8, 8
    arrived, seq0 = make_case(n, f, t, 9, p_loss=0, p_dup=0, p_late=0, n_foreign=0)
    twisted = arrived[0].copy()
    twisted[40:60] ^= 0x5A                                      # same header, other payload bytes
    for order in ([arrived[0], twisted, arrived[1]], [twisted, arrived[0], arrived[1]], [arrived[1], twisted, arrived[0]]):
        pk = np.stack(order)
        want = oa.assemble(pk, n, f, t, seq0)
        assert want["duplicates"] == 1
        check(run_gpu(xb, pk, n, f, t, seq0), want)


def test_nothing_arrives_and_everything_foreign(xb):
    n, f, t = 32, 8, 16
    empty = np.zeros((0, oa.packet_bytes(n, 4, 8)), dtype=np.uint8)
    got = run_gpu(xb, empty, n, f, t, 0)
    check(got, oa.assemble(empty, n, f, t, 0))
    assert got[0].max() == 0 and got[2].tolist() == [t] * f
    arrived, seq0 = make_case(n, f, t, 3, n_foreign=0)
    check(run_gpu(xb, arrived, n, f, t, seq0 + t), oa.assemble(arrived, n, f, t, seq0 + t))   # the next frame's window: all rejected


def test_errors(xb):
    a = xb.Assembler(16, 8, 16)
    fr = torch.empty(16 * 8 * 16 + 16, dtype=torch.uint8, device="cuda")
    pk = torch.empty(a.packet_bytes + 16, dtype=torch.uint8, device="cuda")
    assert xb.xcorr_assemble(a.handle, pk.data_ptr(), 1, 0, 0) == xb.XCORR_EINVAL                 # no frame
    assert xb.xcorr_assemble(a.handle, pk.data_ptr() + 1, 1, 0, fr.data_ptr()) == xb.XCORR_EINVAL  # misaligned packets
    assert xb.xcorr_assemble(a.handle, pk.data_ptr(), 1, 0, fr.data_ptr() + 4) == xb.XCORR_EINVAL  # misaligned frame
    assert xb.xcorr_assemble(a.handle, 0, 1, 0, fr.data_ptr()) == xb.XCORR_EINVAL                  # NULL packets, n > 0
    a.close()


def test_packets_to_normalised_visibilities_end_to_end(xb):
    """assemble -> xcorr_process + xcorr_norm_process_dev (device counters) -> xcorr_read_normalized, two frames, against
    the three oracles chained the same way."""
    n, f, t = 48, 16, 256
    x = xb.XCorr(n, f, t)
    x.norm_enable()
    a = xb.Assembler(n, f, t)
    vis = np.zeros((f, n * (n + 1) // 2, 2), dtype=np.int64)
    flags_all, lost_all = [], np.zeros(f, dtype=np.int64)
    for k in range(2):
        arrived, seq0 = make_case(n, f, t, 50 + 10 * k, kind="gaussian", seq0=10_000 + k * t)
        want = oa.assemble(arrived, n, f, t, seq0)
        frame, flags, lost, _ = a.assemble(torch.from_numpy(arrived.reshape(-1)).cuda(), arrived.shape[0], seq0)
        x.process(frame)
        x.norm_process_dev(flags, lost)
        vis += oracle.planar(want["frame"]).astype(np.int64)
        flags_all.append(np.unpackbits(want["flags"], axis=-1, bitorder="little").astype(bool))
        lost_all += want["lost"]
    L = torch.empty((f, n * (n + 1) // 2), dtype=torch.int32, device="cuda")
    got = x.read_normalized(lost_out=L).cpu().numpy()
    want_L = on.lost_matrix(np.concatenate(flags_all, axis=0), lost_all)
    assert np.array_equal(L.cpu().numpy().astype(np.int64), want_L)
    want_v = on.normalise(vis, 2 * t, want_L)
    assert np.all(np.abs(got - want_v) <= 2.0 ** -22 * np.abs(want_v))
    # the integration has ended: device-side loss counters start again from zero
    frame, flags, lost, _ = a.assemble(None, 0, 0)
    x.process(frame); x.norm_process_dev(flags, None)
    assert int(x.read_normalized(lost_out=L).abs().sum()) == 0 and int(L.sum()) == 0
    a.close(); x.close()


def test_assemble_then_process_with_promise_on_one_stream(xb):
    """xcorr_promise_complete_frames with the frame written by assemble_kernel immediately before xcorr_process on the same
    stream (assemble_kernel never signals early launch completion, so it qualifies): several frames back to back into one
    ring of two frame buffers, every result exact.  Shape with several work segments per worker."""
    n, f, t = 256, 160, 192
    cases = [make_case(n, f, t, 700 + 3 * k, kind="gaussian", seq0=90_000 + k * t) for k in range(4)]
    wants = [oa.assemble(arr, n, f, t, seq0) for arr, seq0 in cases]
    pk = [torch.from_numpy(arr.reshape(-1)).cuda() for arr, _ in cases]
    a = xb.Assembler(n, f, t)
    x = xb.XCorr(n, f, t)
    x.promise_complete_frames()
    st = torch.cuda.Stream()
    bufs = [(torch.empty((t, f, n), dtype=torch.uint8, device="cuda"), torch.empty((t, f, n // 8), dtype=torch.uint8, device="cuda"))
            for _ in range(2)]
    outs = []
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        for k, (arr, seq0) in enumerate(cases):
            frame, flags = bufs[k % 2]
            a.assemble(pk[k], arr.shape[0], seq0, frame=frame, flags=flags, stream=st)
            x.process(frame, st)
            outs.append(x.read(None, st))
    torch.cuda.synchronize()
    for w, o in zip(wants, outs):
        assert np.array_equal(o.cpu().numpy(), oracle.planar(w["frame"]))
    a.close(); x.close()


def test_assemble_accounted_equals_assemble_plus_norm_process(xb):
    """xcorr_assemble_accounted: flags and packet losses counted inside assemble_kernel.  Same L (bit-exact) and the same
    normalised visibilities as the oracles chained; the optional flag field / loss counters it can still write are exact too.
    Dense flags (bursts with many inputs flagged together) so that the O(E^2) intersection path runs, two frames, N with
    several 16-byte footer chunks per sample (272) and with several samples per chunk (16, 48)."""
    for (n, f, t) in [(272, 16, 64), (48, 16, 128), (16, 8, 64)]:
        x = xb.XCorr(n, f, t)
        x.norm_enable()
        a = xb.Assembler(n, f, t)
        vis = np.zeros((f, n * (n + 1) // 2, 2), dtype=np.int64)
        flags_all, lost_all = [], np.zeros(f, dtype=np.int64)
        for k in range(2):
            fr = wl.make_frame("gaussian", n, f, t, 400 + k)
            fl, _, _ = wl.draw_flags_and_loss(n, f, t, 410 + k, p_flag=0.02, p_burst=0.05, burst_frac=0.3, p_packet_loss=0.0)
            pk = wl.packetise(fr, wl.pack_flags(fl), 7_000 + k * t)
            arrived = wl.disturb_packets(pk, 420 + k, p_loss=0.1, p_dup=0.05, p_late=0.1, n_foreign=4)
            want = oa.assemble(arrived, n, f, t, 7_000 + k * t)
            frame, flags, lost, counts = a.assemble(torch.from_numpy(arrived.reshape(-1)).cuda(), arrived.shape[0], 7_000 + k * t,
                                                    account_into=x)
            x.process(frame)
            check((frame.cpu().numpy(), flags.cpu().numpy(), lost.cpu().numpy(), counts.cpu().numpy()), want)
            vis += oracle.planar(want["frame"]).astype(np.int64)
            flags_all.append(np.unpackbits(want["flags"], axis=-1, bitorder="little").astype(bool))
            lost_all += want["lost"]
        L = torch.empty((f, n * (n + 1) // 2), dtype=torch.int32, device="cuda")
        got = x.read_normalized(lost_out=L).cpu().numpy()
        want_L = on.lost_matrix(np.concatenate(flags_all, axis=0), lost_all)
        assert np.array_equal(L.cpu().numpy().astype(np.int64), want_L)
        want_v = on.normalise(vis, 2 * t, want_L)
        assert np.all(np.abs(got - want_v) <= 2.0 ** -22 * np.abs(want_v))
        # the read ended the integration for the accumulators the assembler writes into as well
        frame, _, _, _ = a.assemble(None, 0, 0, account_into=x)
        x.process(frame)
        x.read_normalized(lost_out=L)
        assert (L.cpu().numpy() == t).all()                 # nothing arrived: every sample of every channel lost, no flags
        with pytest.raises(xb.XCorrError):
            a.assemble(None, 0, 0, account_into=xb.XCorr(n, f, t))     # normalisation not enabled on that handle
        a.close(); x.close()


@pytest.mark.parametrize("promise", [False, True])
def test_streamed_packet_path(xb, promise):
    """Pinned packet rings -> xcorr_stream_submit_packets (H2D, assemble, correlate, flag / loss accounting) x 5 frames over a
    depth-2 ring -> one normalised read; and the same stream without normalisation -> exact int32 visibilities."""
    n, f, t = 32, 16, 128
    cases = [make_case(n, f, t, 300 + 7 * k, kind="gaussian", seq0=50_000 + k * t) for k in range(5)]
    wants = [oa.assemble(arr, n, f, t, seq0) for arr, seq0 in cases]
    max_pk = max(arr.shape[0] for arr, _ in cases)
    pinned = [torch.from_numpy(arr.reshape(-1)).pin_memory() for arr, _ in cases]
    vis_sum = sum(oracle.planar(w["frame"]).astype(np.int64) for w in wants)
    for norm in (False, True):
        x = xb.XCorr(n, f, t)
        if promise:
            x.promise_complete_frames()
        if norm:
            x.norm_enable()
        a = xb.Assembler(n, f, t)
        s = xb.XCorrStream(x, depth=2)
        s.attach_assembler(a, max_pk)
        for (arr, seq0), p in zip(cases, pinned):
            s.submit_packets(p, arr.shape[0], seq0)
        if not norm:
            out = torch.empty((f, x.n_pairs, 2), dtype=torch.int32).pin_memory()
            s.read(out)
            assert np.array_equal(out.numpy(), vis_sum)
        else:
            out = torch.empty((f, x.n_pairs, 2), dtype=torch.float32).pin_memory()
            L = torch.empty((f, x.n_pairs), dtype=torch.int32).pin_memory()
            s.read_normalized(out, L)
            flags_all = np.concatenate([np.unpackbits(w["flags"], axis=-1, bitorder="little").astype(bool) for w in wants], axis=0)
            want_L = on.lost_matrix(flags_all, sum(w["lost"] for w in wants))
            assert np.array_equal(L.numpy().astype(np.int64), want_L)
            want_v = on.normalise(vis_sum, 5 * t, want_L)
            assert np.all(np.abs(out.numpy() - want_v) <= 2.0 ** -22 * np.abs(want_v))
        # more packets than the ring slots hold
        assert xb.xcorr_stream_submit_packets(s.stream, pinned[0].data_ptr(), max_pk + 1, 0) == xb.XCORR_EINVAL
        s.close(); a.close(); x.close()


def test_c2_full_size_assembly(xb):
    """BASELINE C2 shape (N=256, F=64, T=16384: 32768 packets of 9248 bytes), the launch configuration bench.py times:
    the whole frame, flag field and counters against what the generator dropped (properties that hold at any size), and
    sampled positions against the oracle run on just their packets."""
    n, f, t, S, C = 256, 64, 16384, 4, 8
    rng = np.random.default_rng(77)
    fr = rng.integers(0, 256, (t, f, n), dtype=np.uint8)
    fb = np.zeros((t, f, n // 8), dtype=np.uint8)
    hit = rng.integers(0, fb.size, 40_000)
    fb.reshape(-1)[hit] = rng.integers(1, 256, hit.size, dtype=np.uint8)
    pk = wl.packetise(fr, fb, 10 ** 12)
    arrived = wl.disturb_packets(pk, 78, p_loss=2e-3, p_dup=1e-3, p_late=5e-3, n_foreign=30)
    frame, flags, lost, counts = run_gpu(xb, arrived, n, f, t, 10 ** 12)
    hdr_seq = arrived[:, 8:16].copy().view("<u8").ravel()
    ok = (arrived[:, 0:4].copy().view("<u4").ravel() == wl.PACKET_MAGIC) & (arrived[:, 4:8].copy().view("<u4").ravel() < f // C) \
        & (hdr_seq >= 10 ** 12) & (hdr_seq < 10 ** 12 + t) & ((hdr_seq - 10 ** 12) % S == 0)
    pos = ((hdr_seq[ok] - 10 ** 12) // S) * (f // C) + arrived[ok, 4:8].copy().view("<u4").ravel()
    present = np.zeros((t // S) * (f // C), dtype=bool)
    present[pos] = True
    assert counts[:3].tolist() == [int(present.sum()), int(ok.sum() - present.sum()), int((~ok).sum())]
    mask = np.repeat(np.repeat(present.reshape(t // S, f // C), S, axis=0), C, axis=1)
    assert np.array_equal(lost, (~mask).sum(axis=0))
    want = fr.copy()
    want[np.unpackbits(fb, axis=-1, bitorder="little").astype(bool)] = 0
    want[~mask] = 0
    assert np.array_equal(frame, want)
    assert np.array_equal(flags, np.where(mask[:, :, None], fb, 0))
    # sampled positions, one by one through the oracle (a 1-block, 1-stream frame holding only that position's packets)
    for p in rng.integers(0, present.size, 12):
        blk, s = divmod(int(p), f // C)
        mine = arrived[ok][pos == p].copy()
        mine[:, 4:8] = 0
        w = oa.assemble(mine, n, C, S, 10 ** 12 + blk * S, S, C)
        assert np.array_equal(frame[blk * S:(blk + 1) * S, s * C:(s + 1) * C], w["frame"])
        assert np.array_equal(flags[blk * S:(blk + 1) * S, s * C:(s + 1) * C], w["flags"])
