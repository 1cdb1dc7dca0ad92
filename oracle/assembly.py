"""CPU ORACLE for packet -> frame assembly -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu legs may import this.  Plain Python loops over
the packets in ARRIVAL order, numpy only for byte slicing; shares nothing with the CUDA path.  It follows PAPER.md
section II-A ("UDP Packet Processing") step by step:

  "All that is required of the system is to place that data into the right location in a large host frame"  (:65)
  "all 256 inputs for one frequency take up 256 bytes.  For 8 frequency bands this represents 2KB.  ...  4 time
   samples are recorded in each packet.  The header contains a streamID that identifies which frequency bands
   are represented in the packet, and a sequence number which gives the relative time"                      (:67)
  "When the system detects packet loss, it writes zeros into the area of the GPU staging buffer where the missing
   packet would have been placed.  ...  the buffer will have good data or zeros in every location.  In the case
   of out of order packets, the sequence number is used to copy the packet into the correct location.
   Duplicate packets are simply ignored."                                                                   (:81)
  "The network threads track packet loss and F-engine error flags" (:113); flags sit in "bit-fields in the packet
   footers" (:116); lost / flagged "data points are zeroed, before they are transferred to the GPU"         (:113)

Readings where the paper is silent (Fig. 3, the packet format, is an image that did not survive; DESIGN.md
section 13, P1..P6):
  P1  wire format of one packet (little endian):  32-byte header {u32 magic 0x58454E47, u32 stream_id, u64 seq,
      16 reserved bytes}, payload uint8[S][C][N] (S = 4 time samples, C = 8 channels; input fastest,
      "can be used by the GPU without modification", :65), footer uint8[S][C][N/8] flag bits (N1).
      For N = 256 that is 9248 bytes ("~9K", :59).
  P2  seq is the array-wide index of the packet's FIRST time sample; a frame starts at sample seq0 and holds
      samples [seq0, seq0 + T).  stream_id s carries channels [C s, C s + C).
  P3  a packet whose magic is wrong, whose stream_id is not below F / C, or whose seq lies outside the frame or
      is not a multiple of S away from seq0, is not part of this frame: it is skipped (counted as rejected).
  P4  duplicates: the FIRST packet in arrival order that claims a (time block, stream) position is kept, later
      ones are ignored -- so the result is defined even if a duplicate's bytes differ.
  P5  the assembler also zeroes the voltage byte of every flagged sample (the paper's "the data points are
      zeroed" does not say where; doing it here makes DESIGN.md N1 hold by construction; it is idempotent).
  P6  the packet-loss counter is kept per channel, lost[f] = S x (missing packets of f's stream)  (N2);
      a lost packet contributes no flags.

Pins (tests/test_oracle_assembly.py): a hand-worked packet stream (tests/golden/assembly.txt); loss-free in-order
packets give back the frame they were cut from; any arrival order gives the same frame; the result equals the
source frame with lost blocks and flagged samples zeroed; lost[f] + S x (packets kept for f) = T.
"""
from __future__ import annotations

import struct

import numpy as np

MAGIC = 0x58454E47
HEADER_BYTES = 32


def packet_bytes(n_inputs: int, s_per_packet: int, c_per_packet: int) -> int:
    """P1: header + payload + flag footer."""
    return HEADER_BYTES + s_per_packet * c_per_packet * n_inputs + s_per_packet * c_per_packet * n_inputs // 8


def parse_header(pkt: bytes):
    """P1: (magic, stream_id, seq) of one packet."""
    magic, stream_id, seq = struct.unpack_from("<IIQ", pkt, 0)
    return magic, stream_id, seq


def assemble(packets, n_inputs: int, n_freq: int, n_time: int, seq0: int, s_per_packet: int = 4, c_per_packet: int = 8):
    """Walk the packets in arrival order and build one frame.

    packets : iterable of bytes-like, each packet_bytes() long, in the order they arrived.
    Returns dict(frame uint8[T][F][N], flags uint8[T][F][N/8] (wire bit-field), lost int64[F],
                 kept, duplicates, rejected : packet counts).
    """
    S, C, N = s_per_packet, c_per_packet, n_inputs
    assert n_time % S == 0 and n_freq % C == 0 and N % 8 == 0
    n_streams = n_freq // C
    pbytes = packet_bytes(N, S, C)
    # "the buffer will have good data or zeros in every location": start from zeros, i.e. every position is "lost"
    frame = np.zeros((n_time, n_freq, N), dtype=np.uint8)
    flags = np.zeros((n_time, n_freq, N // 8), dtype=np.uint8)
    seen = set()
    kept = duplicates = rejected = 0
    for pkt in packets:
        pkt = bytes(pkt)
        assert len(pkt) == pbytes
        magic, stream_id, seq = parse_header(pkt)
        # P3: not a packet of this frame
        if magic != MAGIC or stream_id >= n_streams or seq < seq0 or seq >= seq0 + n_time or (seq - seq0) % S != 0:
            rejected += 1
            continue
        t0 = seq - seq0
        where = (t0 // S, stream_id)
        # "Duplicate packets are simply ignored." (P4: first arrival wins)
        if where in seen:
            duplicates += 1
            continue
        seen.add(where)
        kept += 1
        # "the sequence number is used to copy the packet into the correct location"
        payload = np.frombuffer(pkt, dtype=np.uint8, count=S * C * N, offset=HEADER_BYTES).reshape(S, C, N)
        footer = np.frombuffer(pkt, dtype=np.uint8, count=S * C * N // 8, offset=HEADER_BYTES + S * C * N).reshape(S, C, N // 8)
        # P5: a flagged sample's voltage byte is zero in the frame; input n is bit n % 8 of footer byte n // 8 (N1)
        flagged = np.zeros((S, C, N), dtype=bool)
        for n in range(N):
            flagged[:, :, n] = (footer[:, :, n // 8] >> (n % 8)) & 1
        data = payload.copy()
        data[flagged] = 0
        for dt in range(S):
            frame[t0 + dt, C * stream_id:C * stream_id + C] = data[dt]
            flags[t0 + dt, C * stream_id:C * stream_id + C] = footer[dt]
    # P6: packet loss, per channel, in time samples
    lost = np.zeros(n_freq, dtype=np.int64)
    for blk in range(n_time // S):
        for s in range(n_streams):
            if (blk, s) not in seen:
                lost[C * s:C * s + C] += S
    return {"frame": frame, "flags": flags, "lost": lost, "kept": kept, "duplicates": duplicates, "rejected": rejected}
