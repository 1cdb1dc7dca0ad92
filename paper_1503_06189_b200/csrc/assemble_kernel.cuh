// assemble_kernel.cuh -- packet -> frame assembly (SURVEY.md 8(f) NEXT-2; section II-A, :59-:81).
//
// The paper's network threads place each UDP payload "into the right location in a large host frame" (:65) by its
// sequence number, write zeros where a packet is missing, and ignore duplicates (:81).  Here that is two kernels over
// the packets as they arrived (wire format: include/xcorr_assemble.h, P1):
//
//   packet_claim_kernel   one thread per packet: parse the header, reject what is not of this frame (P3), and claim the
//                         packet's position (time block, stream) with atomicMin(arrival index) -- the first arrival
//                         wins whatever the order in which threads run (P4), out-of-order packets need nothing else.
//   assemble_kernel       one pass over the POSITIONS of the frame (grid-stride, one CTA per position at a time): copy
//                         the owner's payload as 16-byte vectors into the S rows of the frame, zeroing the byte of every
//                         flagged sample (P5) -- the footer is "read initially as 32-bit integers, and bit-field
//                         extraction is performed only if ... non-zero": here 16 flag bits per 16 voltage
//                         bytes, expanded only when non-zero; copy the footer into the frame's flag bit-field; where no
//                         packet owns the position write zeros ("good data or zeros in every location", :81) and add S to
//                         the channels' packet-loss counters (:113, P6).  Every byte of the frame and of the flag field
//                         is written exactly once: no clearing pass.
//
//                         With kAccount (xcorr_assemble_accounted) the same pass also does the flag / loss accounting of
//                         the lost-sample normalisation (normalise_kernel.cuh; PAPER.md:113-:123): every footer word is in
//                         a register here anyway, so a non-zero one is expanded on the spot into the handle's intersection /
//                         counter accumulator X, and the loss counters go straight into the handle's -- the flag field need
//                         not be written to memory and read back by flag_count_kernel at all.
//
// HBM-bound: per frame, reads n_packets * packet_bytes, writes T*F*N (+ T*F*N/8 if the flag field is wanted).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.hpp"
#include "normalise_kernel.cuh"

namespace xc {

constexpr uint32_t kPacketMagic = 0x58454E47u;
constexpr int kPacketHeaderBytes = 32;
constexpr uint32_t kNoOwner = 0xFFFFFFFFu;

struct AssembleShape {
    int n_inputs, n_freq, n_time;   // N, F, T
    int s_per_packet, c_per_packet; // S, C
    int n_streams, n_blocks;        // F / C, T / S
    unsigned long long packet_bytes;
};

// counts[0] kept  [1] duplicates  [2] rejected  [3] positions lost  [4] valid (scratch)  [5] CTA ticket (scratch)
// The ownership table and the counters are all-kNoOwner / all-zero on entry (no memset between calls): there are two
// tables used alternately, assemble_kernel resets the one the previous frame used while it reads this frame's, and its
// last CTA zeroes the counters.  `lost` (caller's int32[F]) is zeroed here.
__global__ void __launch_bounds__(256) packet_claim_kernel(const uint8_t *__restrict__ packets, unsigned int n_packets,
                                                            unsigned long long seq0, AssembleShape sh, uint32_t *__restrict__ owner,
                                                            uint32_t *__restrict__ counts, int32_t *__restrict__ lost)
{
    const unsigned int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (lost && k < (unsigned)sh.n_freq) lost[k] = 0;
    bool valid = false, rejected = false;
    if (k < n_packets) {
        const uint4 hdr = __ldg(reinterpret_cast<const uint4 *>(packets + (unsigned long long)k * sh.packet_bytes));
        const uint32_t magic = hdr.x, stream = hdr.y;
        const unsigned long long seq = (unsigned long long)hdr.z | ((unsigned long long)hdr.w << 32);
        const unsigned long long dt = seq - seq0;     // wraps for seq < seq0 -> fails the range test
        valid = magic == kPacketMagic && stream < (uint32_t)sh.n_streams && seq >= seq0 && dt < (unsigned long long)sh.n_time &&
                dt % (unsigned)sh.s_per_packet == 0;
        rejected = !valid;
        if (valid) atomicMin(owner + (dt / (unsigned)sh.s_per_packet) * (unsigned)sh.n_streams + stream, k);
    }
    // warp-aggregated counters
    const unsigned v = __ballot_sync(0xFFFFFFFFu, valid), r = __ballot_sync(0xFFFFFFFFu, rejected);
    if ((threadIdx.x & 31) == 0) {
        if (v) atomicAdd(counts + 4, __popc(v));
        if (r) atomicAdd(counts + 2, __popc(r));
    }
}

// 4 flag bits -> 4 byte masks (0xFF where flagged): bit k of x goes to bit 8k (the partial products never collide)
__device__ __forceinline__ uint32_t spread4(uint32_t x) { return (((x & 0xFu) * 0x00204081u) & 0x01010101u) * 0xFFu; }

// kAccount, the rare path: some lanes of the warp hold footer chunks (16 bytes = 128 flag bits each, chunk cw + lane of the
// position) with flags set (mask nz).  "read initially as 32-bit integers, and bit-field extraction is performed only if ...
// non-zero" (:123): c_f[n] += 1 for every flagged input n and X[f][p(n, j)] += 1 for every input j > n flagged in the same
// sample -- the paper's O(E^2) intersection tracking (:117-:119), each flagged bit handled by the whole warp
// (flag_row_update_warp scans the sample's bit-field with one load per lane).  Not inlined: keeps the copy loop at 32 registers.
__device__ __noinline__ void account_flagged_chunks(uint32_t nz, const uint4 v, unsigned cw, unsigned frow_chunks, const uint8_t *__restrict__ foot,
                                                    int N, int C, int f_base, int32_t *__restrict__ x, int32_t *__restrict__ cnt)
{
    const int lane = (int)(threadIdx.x & 31u);
    const long long n_pairs = (long long)N * (N + 1) / 2;
    while (nz) {
        const int src = __ffs((int)nz) - 1;
        nz &= nz - 1;
        const unsigned cs = cw + (unsigned)src;
        const unsigned dts = cs / frow_chunks, ws = cs - dts * frow_chunks;
        const uint8_t *row_bits = foot + (size_t)dts * ((size_t)(C * N) >> 3);      // the footer bytes of time sample dts
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint32_t mine = (q == 0) ? v.x : (q == 1) ? v.y : (q == 2) ? v.z : v.w;
            uint32_t m = __shfl_sync(0xFFFFFFFFu, mine, src);
            while (m) {                                              // warp-uniform
                const int b = __ffs((int)m) - 1;
                m &= m - 1;
                const unsigned idx = ws * 128u + 32u * (unsigned)q + (unsigned)b;     // bit index inside the row
                const int ch = (int)(idx / (unsigned)N), n = (int)(idx % (unsigned)N);
                flag_row_update_warp(reinterpret_cast<const uint16_t *>(row_bits + (size_t)ch * (size_t)(N >> 3)), N, n,
                                     x + (size_t)(f_base + ch) * (size_t)n_pairs, cnt + (size_t)(f_base + ch) * (size_t)N, lane);
            }
        }
    }
}

// kAccount = false: xcorr_assemble.  kAccount = true: xcorr_assemble_accounted -- `x` = the handle's intersection / counter
// accumulator int32[F][P], `cnt` = its flag counters int32[F][N], `lost_acc` = its per-channel loss counters (all added to).
template <bool kAccount>
__global__ void __launch_bounds__(256, 6) assemble_kernel(const uint8_t *__restrict__ packets, AssembleShape sh,
                                                        const uint32_t *__restrict__ owner, uint32_t *__restrict__ owner_next,
                                                        uint8_t *__restrict__ frame,
                                                        uint8_t *__restrict__ flags, int32_t *__restrict__ lost, uint32_t *__restrict__ counts,
                                                        uint32_t *__restrict__ counts_out, int32_t *__restrict__ x, int32_t *__restrict__ cnt,
                                                        int32_t *__restrict__ lost_acc)
{
    const int N = sh.n_inputs, F = sh.n_freq, S = sh.s_per_packet, C = sh.c_per_packet;
    const unsigned row_chunks = (unsigned)(C * N) >> 4;            // 16-byte vectors per time sample of one stream
    const unsigned pay_chunks = row_chunks * (unsigned)S;
    const unsigned frow_chunks = (unsigned)(C * N) >> 7;           // same for the flag bit-field (C*N/8 bytes per sample)
    const unsigned foot_chunks = frow_chunks * (unsigned)S;
    const unsigned long long pay_bytes = (unsigned long long)S * C * N;
    const unsigned n_pos = (unsigned)sh.n_blocks * (unsigned)sh.n_streams;
    uint32_t kept_local = 0, lost_local = 0;                      // thread 0's tallies of this CTA
    for (unsigned pos = blockIdx.x; pos < n_pos; pos += gridDim.x) {
        const unsigned blk = pos / (unsigned)sh.n_streams, stream = pos % (unsigned)sh.n_streams;
        const uint32_t own = __ldg(owner + pos);
        if (threadIdx.x == 0) owner_next[pos] = kNoOwner;          // the table the NEXT frame's claims go to (last frame's, dirty)
        // byte offset of (t = blk*S, f = C*stream, n = 0) in the frame; rows of one stream are C*N contiguous bytes, F*N apart
        const unsigned long long f0 = ((unsigned long long)blk * S * F + (unsigned long long)C * stream) * (unsigned long long)N;
        uint4 *frame_v = reinterpret_cast<uint4 *>(frame + f0);
        const unsigned long long frame_row_stride = ((unsigned long long)F * N) >> 4;   // in uint4
        if (own != kNoOwner) {
            const uint8_t *pkt = packets + (unsigned long long)own * sh.packet_bytes;
            const uint4 *pay = reinterpret_cast<const uint4 *>(pkt + kPacketHeaderBytes);
            const uint16_t *foot16 = reinterpret_cast<const uint16_t *>(pkt + kPacketHeaderBytes + pay_bytes);
            // two vectors per thread in flight (both loads issued before the first store)
            for (unsigned c0 = threadIdx.x; c0 < pay_chunks; c0 += 2 * blockDim.x) {
                const unsigned c1 = c0 + blockDim.x;
                const bool two = c1 < pay_chunks;
                uint4 v0 = __ldg(pay + c0), v1 = make_uint4(0, 0, 0, 0);
                const uint32_t bits0 = __ldg(foot16 + c0);         // the 16 flag bits of these 16 inputs
                uint32_t bits1 = 0;
                if (two) {
                    v1 = __ldg(pay + c1);
                    bits1 = __ldg(foot16 + c1);
                }
                if (bits0 | bits1) {                               // rare: zero the flagged samples' bytes (P5)
                    v0.x &= ~spread4(bits0);       v0.y &= ~spread4(bits0 >> 4);
                    v0.z &= ~spread4(bits0 >> 8);  v0.w &= ~spread4(bits0 >> 12);
                    v1.x &= ~spread4(bits1);       v1.y &= ~spread4(bits1 >> 4);
                    v1.z &= ~spread4(bits1 >> 8);  v1.w &= ~spread4(bits1 >> 12);
                }
                const unsigned dt0 = c0 / row_chunks, w0 = c0 - dt0 * row_chunks;
                frame_v[dt0 * frame_row_stride + w0] = v0;
                if (two) {
                    const unsigned dt1 = c1 / row_chunks, w1 = c1 - dt1 * row_chunks;
                    frame_v[dt1 * frame_row_stride + w1] = v1;
                }
            }
            if (flags || kAccount) {
                const uint4 *foot = reinterpret_cast<const uint4 *>(foot16);
                uint4 *flags_v = reinterpret_cast<uint4 *>(flags + (f0 >> 3));
                // the footer of a position is one warp's job, and the job rotates among the CTA's warps from position to position
                // (the warps run through the position loop independently, so the flag work spreads over all of them)
                const unsigned lane = threadIdx.x & 31u, n_warps = blockDim.x >> 5;
                const unsigned duty = ((threadIdx.x >> 5) + n_warps - (pos / gridDim.x) % n_warps) % n_warps;   // 0 for this position's warp
                for (unsigned cw = duty * 32u; cw < foot_chunks; cw += 32u * n_warps) {     // warp-uniform loop
                    const unsigned c = cw + lane;
                    uint4 v = make_uint4(0, 0, 0, 0);
                    if (c < foot_chunks) {
                        const unsigned dt = c / frow_chunks, w = c - dt * frow_chunks;
                        v = __ldg(foot + c);
                        if (flags) flags_v[dt * (frame_row_stride >> 3) + w] = v;
                    }
                    if constexpr (kAccount) {
                        const uint32_t nz = __ballot_sync(0xFFFFFFFFu, (v.x | v.y | v.z | v.w) != 0);
                        if (nz) account_flagged_chunks(nz, v, cw, frow_chunks, reinterpret_cast<const uint8_t *>(foot), N, C, C * (int)stream, x, cnt);
                    }
                }
            }
            kept_local += 1;
        } else {
            // "it writes zeros into the area of the GPU staging buffer where the missing packet would have been placed" (:81)
            const uint4 z = make_uint4(0, 0, 0, 0);
            for (unsigned c = threadIdx.x; c < pay_chunks; c += blockDim.x) {
                const unsigned dt = c / row_chunks, w = c - dt * row_chunks;
                frame_v[dt * frame_row_stride + w] = z;
            }
            if (flags) {
                uint4 *flags_v = reinterpret_cast<uint4 *>(flags + (f0 >> 3));
                for (unsigned c = threadIdx.x; c < foot_chunks; c += blockDim.x) {
                    const unsigned dt = c / frow_chunks, w = c - dt * frow_chunks;
                    flags_v[dt * (frame_row_stride >> 3) + w] = z;
                }
            }
            if (lost && threadIdx.x < (unsigned)C) atomicAdd(lost + C * stream + threadIdx.x, S);   // packet-loss counter (P6)
            if constexpr (kAccount) {
                if (threadIdx.x < (unsigned)C) atomicAdd(lost_acc + C * stream + threadIdx.x, S);
            }
            lost_local += 1;
        }
    }
    // packet counts: one atomic per CTA; the last CTA to finish derives duplicates = valid - kept, hands the four
    // numbers to the caller and zeroes the scratch for the next frame
    if (threadIdx.x == 0) {
        if (kept_local) atomicAdd(counts + 0, kept_local);
        if (lost_local) atomicAdd(counts + 3, lost_local);
        __threadfence();
        if (atomicAdd(counts + 5, 1u) == gridDim.x - 1) {
            __threadfence();
            const uint32_t kept = atomicExch(counts + 0, 0u), valid = atomicExch(counts + 4, 0u);
            const uint32_t rejected = atomicExch(counts + 2, 0u), lost_pos = atomicExch(counts + 3, 0u);
            counts[5] = 0;
            if (counts_out) {
                counts_out[0] = kept; counts_out[1] = valid - kept; counts_out[2] = rejected; counts_out[3] = lost_pos;
            }
        }
    }
}

// lost-sample counters (one frame's, or the host-side tallies of an integration) -> the handle's device accumulator
// (xcorr_norm_process_dev, xcorr_read_normalized).  `src` may be device memory or page-locked host memory read in place.
__global__ void lost_add_kernel(const int32_t *__restrict__ src, int32_t *__restrict__ lost_acc, int n_freq)
{
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f < n_freq) lost_acc[f] += src[f];
}

}  // namespace xc
