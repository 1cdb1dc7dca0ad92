"""Pins of the packet -> frame assembly oracle (oracle/assembly.py) against things other than itself."""
from pathlib import Path

import numpy as np
import pytest

import oracle.assembly as oa
import workloads as wl

GOLDEN = Path(__file__).parent / "golden" / "assembly.txt"


def load_golden():
    pk, order, rows, lost, counts = {}, [], [], None, None
    for ln in GOLDEN.read_text().splitlines():
        if not ln or ln.startswith("#"):
            continue
        tag, rest = ln.split(None, 1)
        if tag == "P":
            name, rest = rest.split(None, 1)
            hdr, pay, foot = [bytes.fromhex(x.replace(" ", "")) for x in rest.split("|")]
            pk[name] = hdr + bytes(16) + pay + foot
        elif tag == "ORDER":
            order = rest.split()
        elif tag == "R":
            t, f, volt, flag = rest.split()
            rows.append((int(t), int(f), bytes.fromhex(volt), bytes.fromhex(flag)))
        elif tag == "LOST":
            lost = [int(x) for x in rest.split()]
        elif tag == "COUNTS":
            counts = [int(x) for x in rest.split()]
    return pk, order, rows, lost, counts


def test_handworked_packet_stream():
    pk, order, rows, lost, counts = load_golden()
    assert all(len(p) == 68 == oa.packet_bytes(8, 2, 2) for p in pk.values())
    r = oa.assemble([pk[k] for k in order], n_inputs=8, n_freq=4, n_time=4, seq0=100, s_per_packet=2, c_per_packet=2)
    assert len(rows) == 16
    for t, f, volt, flag in rows:
        assert r["frame"][t, f].tobytes() == volt, (t, f)
        assert r["flags"][t, f].tobytes() == flag, (t, f)
    assert r["lost"].tolist() == lost
    assert [r["kept"], r["duplicates"], r["rejected"]] == counts


def test_handworked_first_arrival_wins():
    """Swap A and its differing duplicate C: now C's bytes (0xEE, all flagged -> zeroed) own the position."""
    pk, order, rows, lost, counts = load_golden()
    r = oa.assemble([pk[k] for k in "CBADEFG"], 8, 4, 4, 100, 2, 2)
    assert r["frame"][2:4, 2:4].max() == 0                      # every sample of C is flagged (footer FF) -> zero (P5)
    assert r["flags"][2:4, 2:4].tolist() == [[[0xFF], [0xFF]], [[0xFF], [0xFF]]]
    assert [r["kept"], r["duplicates"], r["rejected"]] == counts


def test_packet_size_matches_the_paper():
    # "Each UDP packet is ~9K in size"; payload 4 x 8 x 256 = 8 KiB (:67); Table I (:139-:140): headers and
    # flags add 7.45 / 6.4 - 1 = 16.4 % = 1344 bytes on the wire, of which the 1024-byte flag footer is part
    assert oa.packet_bytes(256, 4, 8) == 32 + 8192 + 1024 == 9248
    assert 8192 * (7.45 / 6.4 - 1) > 1024 + 32


def _case(n, f, t, seed, **kw):
    fr = wl.uniform_frame(n, f, t, seed)
    flags, _, _ = wl.draw_flags_and_loss(n, f, t, seed + 1, p_flag=0.01, p_burst=0.02, burst_frac=0.2, p_packet_loss=0.0)
    fb = wl.pack_flags(flags)
    return fr, flags, fb, wl.packetise(fr, fb, seq0=5000, **kw)


@pytest.mark.parametrize("n,f,t", [(16, 8, 8), (48, 16, 32), (256, 8, 16)])
def test_lossless_in_order_round_trip(n, f, t):
    fr, flags, fb, pk = _case(n, f, t, 11)
    r = oa.assemble(pk, n, f, t, 5000)
    want = fr.copy()
    want[flags] = 0                                             # P5
    assert np.array_equal(r["frame"], want) and np.array_equal(r["flags"], fb)
    assert r["lost"].tolist() == [0] * f and r["kept"] == pk.shape[0] and r["duplicates"] == r["rejected"] == 0
    # without flags the payload lands unmodified ("can be used by the GPU without modification")
    r0 = oa.assemble(wl.packetise(fr, np.zeros_like(fb), 5000), n, f, t, 5000)
    assert np.array_equal(r0["frame"], fr)


def test_arrival_order_does_not_matter_without_duplicates():
    n, f, t = 32, 16, 64
    fr, flags, fb, pk = _case(n, f, t, 21)
    ref = oa.assemble(pk, n, f, t, 5000)
    rng = np.random.default_rng(5)
    for _ in range(3):
        r = oa.assemble(pk[rng.permutation(pk.shape[0])], n, f, t, 5000)
        assert np.array_equal(r["frame"], ref["frame"]) and np.array_equal(r["flags"], ref["flags"])


def test_loss_duplicates_reordering_equal_the_source_with_lost_blocks_zeroed():
    """'assembled frame == reference frame with lost blocks zeroed', computed here directly from which
    packets were dropped (not through the oracle)."""
    n, f, t, S, C = 32, 16, 128, 4, 8
    fr, flags, fb, pk = _case(n, f, t, 31)
    rng = np.random.default_rng(7)
    drop = rng.random(pk.shape[0]) < 0.15
    arrived = pk[~drop]
    arrived = np.concatenate([arrived, arrived[::5]])           # duplicates (identical bytes), arriving late
    arrived = arrived[rng.permutation(arrived.shape[0])]        # any order
    r = oa.assemble(arrived, n, f, t, 5000)
    want, want_fb, want_lost = fr.copy(), fb.copy(), np.zeros(f, dtype=np.int64)
    want[flags] = 0
    for k in np.nonzero(drop)[0]:
        blk, s = divmod(int(k), f // C)
        want[blk * S:(blk + 1) * S, s * C:(s + 1) * C] = 0       # "it writes zeros into the area ... where the missing packet would have been"
        want_fb[blk * S:(blk + 1) * S, s * C:(s + 1) * C] = 0
        want_lost[s * C:(s + 1) * C] += S
    assert np.array_equal(r["frame"], want) and np.array_equal(r["flags"], want_fb)
    assert np.array_equal(r["lost"], want_lost)
    assert r["kept"] == int((~drop).sum()) and r["duplicates"] == len(arrived) - r["kept"] and r["rejected"] == 0
    # lost[f] + S x (packets kept for f's stream) = T
    kept_per_stream = np.bincount(np.nonzero(~drop)[0] % (f // C), minlength=f // C)
    assert np.array_equal(r["lost"] + S * np.repeat(kept_per_stream, C), np.full(f, t))


def test_foreign_packets_are_rejected_and_other_frames_ignored():
    n, f, t = 16, 8, 16
    fr, flags, fb, pk = _case(n, f, t, 41)
    ref = oa.assemble(pk, n, f, t, 5000)
    arrived = wl.disturb_packets(pk, 9, p_loss=0.0, p_dup=0.0, p_late=0.0, n_foreign=6)
    r = oa.assemble(arrived, n, f, t, 5000)
    assert r["rejected"] == 6 and np.array_equal(r["frame"], ref["frame"])
    # the same packets seen by the NEXT frame's assembler: none belongs to it
    r2 = oa.assemble(pk, n, f, t, 5000 + t)
    assert r2["kept"] == 0 and r2["rejected"] == pk.shape[0] and r2["frame"].max() == 0 and r2["lost"].tolist() == [t] * f


def test_nothing_arrives_everything_lost():
    r = oa.assemble([], 16, 8, 8, 0)
    assert r["frame"].max() == 0 and r["lost"].tolist() == [8] * 8


def test_generator_disturb_statistics():
    n, f, t = 16, 8, 4096
    fr, flags, fb, pk = _case(n, f, t, 51)
    arrived = wl.disturb_packets(pk, 3, p_loss=0.05, p_dup=0.05, p_late=0.1)
    r = oa.assemble(arrived, n, f, t, 5000)
    assert abs(1 - r["kept"] / pk.shape[0] - 0.05) < 0.02 and abs(r["duplicates"] / pk.shape[0] - 0.0475) < 0.02
    seqs = arrived[:, 8:16].copy().view("<u8").ravel()
    assert (np.diff(seqs.astype(np.int64)) < 0).any()           # some packets really are out of order
