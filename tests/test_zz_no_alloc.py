"""xcorr_assemble_static -- packet -> frame assembly for callers that must not allocate (include/xcorr_assemble.h).

Who that is: the per-frame threads of a running acquisition (nothing is allocated outside start-up and
shutdown -- a cudaMalloc from any thread stalls every stream of the device in the middle of an integration), and
processes whose device memory another allocator already owns.  For them the ownership tables and counters that
xcorr_assembler_create() gets from cudaMalloc live in a fixed array inside libxcorr.so instead.

What is checked here: the new entry point gives byte for byte what the existing path (an xcorr_assembler handle and
xcorr_assemble) gives on the same packets -- frame, flag field, loss counters, packet counts; assembly is byte work, so
the tolerance is the one the other assembly tests use: none -- on two calls in a row whose shapes differ, so that the
second call meets whatever the first left in the shared array; that the second call leaves the device's free memory
where it was; and that a frame beyond the array's fixed capacity is refused, not grown into.

This file is named to be collected last: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  It passes run alone in a fresh process (the entry point's first call then also does its one-time
per-device set-up) and run after everything else (the library's device code is then already loaded).
"""
import numpy as np
import pytest

import oracle.assembly as oa
import workloads as wl

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def xb():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1503_06189_b200 as xb
    return xb


def arrivals(n, f, t, seed, S, C, seq0):
    """Packets of one synthetic frame as they arrive: some lost, some twice, some late, a few of another frame."""
    fr = wl.make_frame("uniform", n, f, t, seed)
    flags, _, _ = wl.draw_flags_and_loss(n, f, t, seed + 1, p_flag=5e-3, p_burst=5e-3, burst_frac=0.1, p_packet_loss=0.0)
    pk = wl.packetise(fr, wl.pack_flags(flags), seq0, S, C)
    return wl.disturb_packets(pk, seed + 2, p_loss=0.15, p_dup=0.1, p_late=0.2, n_foreign=5)


def outputs(n, f, t, poison):
    """Caller-owned outputs, pre-filled so that a byte the kernels fail to write shows."""
    return (torch.full((t, f, n), poison, dtype=torch.uint8, device="cuda"),
            torch.full((t, f, n // 8), poison, dtype=torch.uint8, device="cuda"),
            torch.full((f,), -7, dtype=torch.int32, device="cuda"),
            torch.full((4,), -7, dtype=torch.int32, device="cuda"))


def existing_path(xb, pk_dev, n_packets, n, f, t, S, C, seq0):
    a = xb.Assembler(n, f, t, S, C)
    frame, flags, lost, counts = outputs(n, f, t, 0xA5)
    a.assemble(pk_dev if n_packets else None, n_packets, seq0, frame=frame, flags=flags, lost=lost, counts=counts)
    torch.cuda.synchronize()
    a.close()
    return frame, flags, lost, counts


def static_path(xb, pk_dev, n_packets, n, f, t, S, C, seq0, out):
    frame, flags, lost, counts = out
    rc = xb.xcorr_assemble_static(n, f, t, S, C, pk_dev.data_ptr() if n_packets else 0, n_packets, seq0, frame.data_ptr(),
                                  flags.data_ptr(), lost.data_ptr(), counts.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert rc == xb.XCORR_OK, (xb.xcorr_strerror(rc), xb.xcorr_assemble_static_last_cuda_error())


def same(got, want):
    for g, w in zip(got, want):
        assert torch.equal(g, w)


def test_static_entry_point_matches_the_allocating_path_twice_in_a_row(xb):
    # two frames of different shape: the first uses 1024 positions of the shared table, the second 170 of them with
    # other packet sizes -- it starts on the first call's leftovers (owners, counters) and must not see them
    shapes = [(256, 64, 512, 4, 8, 1_000_000), (144, 40, 68, 2, 8, 77)]
    cases = []
    for k, (n, f, t, S, C, seq0) in enumerate(shapes):
        arr = arrivals(n, f, t, 900 + k, S, C, seq0)
        cases.append((arr, torch.from_numpy(arr.reshape(-1)).cuda(), outputs(n, f, t, 0x5A)))
    wants = [existing_path(xb, pk, arr.shape[0], n, f, t, S, C, seq0) for (arr, pk, _), (n, f, t, S, C, seq0) in zip(cases, shapes)]
    torch.cuda.synchronize()

    # first call on this device (does the one-time set-up if no earlier test did), then the second straight behind it on
    # the same stream with no synchronisation in between
    free_before = None
    for k, ((arr, pk, out), (n, f, t, S, C, seq0)) in enumerate(zip(cases, shapes)):
        if k == 1:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
        static_path(xb, pk, arr.shape[0], n, f, t, S, C, seq0, out)
    torch.cuda.synchronize()
    # the second call took nothing from the device: free memory as the driver reports it has not moved
    assert torch.cuda.mem_get_info()[0] == free_before
    for (arr, pk, out), want in zip(cases, wants):
        same(out, want)

    # and both agree with the CPU oracle, so "equal" is not "equally wrong"
    for (arr, pk, out), (n, f, t, S, C, seq0) in zip(cases, shapes):
        ref = oa.assemble(arr, n, f, t, seq0, S, C)
        assert np.array_equal(out[0].cpu().numpy(), ref["frame"]) and np.array_equal(out[1].cpu().numpy(), ref["flags"])
        assert np.array_equal(out[2].cpu().numpy().astype(np.int64), ref["lost"])
        assert out[3].cpu().numpy()[:3].tolist() == [ref["kept"], ref["duplicates"], ref["rejected"]]

    # the same frame again, and an empty one (nothing arrived: all zeros, every sample lost), back to back
    (arr, pk, _), (n, f, t, S, C, seq0) = cases[1], shapes[1]
    again, empty = outputs(n, f, t, 0x3C), outputs(n, f, t, 0x3C)
    static_path(xb, pk, arr.shape[0], n, f, t, S, C, seq0, again)
    static_path(xb, pk, 0, n, f, t, S, C, seq0, empty)
    torch.cuda.synchronize()
    same(again, wants[1])
    assert int(empty[0].max()) == 0 and int(empty[1].max()) == 0 and empty[2].tolist() == [t] * f
    assert empty[3].tolist() == [0, 0, 0, (t // S) * (f // C)]


def test_static_entry_point_refuses_what_its_table_cannot_hold(xb):
    n, S, C = 16, 1, 8
    cap = xb.XCORR_ASSEMBLE_STATIC_MAX_POSITIONS
    frame = torch.zeros(1024, dtype=torch.uint8, device="cuda")
    # (T / S) * (F / C) = cap + 1 positions: refused before anything is enqueued (the tiny frame buffer is never touched)
    rc = xb.xcorr_assemble_static(n, 8, cap + 1, S, C, 0, 0, 0, frame.data_ptr())
    assert rc == xb.XCORR_ELIMIT and "scratch" in xb.xcorr_strerror(rc)
    torch.cuda.synchronize()
    assert int(frame.max()) == 0
    # the shape rules of xcorr_assembler_create hold here too
    assert xb.xcorr_assemble_static(n, 8, 16, 3, C, 0, 0, 0, frame.data_ptr()) == xb.XCORR_EINVAL      # T % S != 0
    assert xb.xcorr_assemble_static(n, 8, 16, 4, C, 0, 0, 0, 0) == xb.XCORR_EINVAL                      # no frame
    assert xb.xcorr_assemble_static(n, 8, 16, 4, C, 0, 0, 0, frame.data_ptr() + 4) == xb.XCORR_EINVAL  # misaligned frame
    # exactly at capacity is accepted
    t = cap
    big = torch.full((t * 8 * n,), 0x77, dtype=torch.uint8, device="cuda")
    assert xb.xcorr_assemble_static(n, 8, t, S, C, 0, 0, 0, big.data_ptr()) == xb.XCORR_OK
    torch.cuda.synchronize()
    assert int(big.max()) == 0
