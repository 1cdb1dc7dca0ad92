// normalise_kernel.cuh -- lost-sample normalisation (section II-C).
//
// The paper's post-processing thread builds, per integration, a normalisation matrix from a packet-loss counter
// (added to every point, :115), per-(input, frequency) F-engine flag counters (:116) and the per-sample
// intersections of inputs flagged together (subtracted, :117-119), and applies the lost fraction to the
// correlation matrix (:121).  Here the flag bit-fields of every frame are reduced on the GPU by
// flag_count_kernel into ONE accumulator
//
//     X[f][p(i,j)] = number of samples of channel f in which inputs i and j were both flagged   (i <= j)
//
// whose diagonal X[f][p(i,i)] is the flag counter c_f[i]; xcorr_read_normalized's finalize pass then forms
//
//     L[f][i,j] = lost[f] + X_ii + X_jj - X_ij   (i != j),     L[f][i,i] = lost[f] + X_ii          (N2, N3)
//     V~[f][i,j] = V[f][i,j] * T / (T - L[f][i,j])   in float32, 0 where T - L <= 0                (N4, N5)
//
// fused into the packed-triangle write of finalize_kernel (finalize_kernel.cuh, kNormalise = true).
//
// Flag wire format (N1): uint8[T][F][N/8], input n of sample (t, f) is bit (n % 8) of byte n / 8.
// "the bit-field of flags in the footer is read initially as 32-bit integers, and bit-field extraction is performed
// only if the 32-bit representation of the bit-field is non-zero": a warp reads 2 KiB of bit-field per
// iteration (4 x 128 bits per lane, coalesced) and goes on at once if all of it is zero; each set bit is then handled
// by the whole warp (the row scan is one load per lane), the per-sample intersection work is O(E^2) as in the paper.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.hpp"

namespace xc {

// One flagged bit (sample s, input n), handled by a whole warp: add 1 to the counter c_f[n] and to X[f][p(n, j)] for every
// input j > n flagged in the same sample.  The sample's bit-field is n_inputs / 16 aligned halfwords; lane l takes halfwords
// (n >> 4) + l, + 32, ... so the row is scanned with one (L1-resident) load per lane.
__device__ __forceinline__ void flag_row_update_warp(const uint16_t *__restrict__ sample_bits, int n_inputs, int n, int32_t *x_f,
                                                     int32_t *cnt_f, int lane)
{
    const int n_half = n_inputs >> 4;
    const long long row = pair_index(n_inputs, n, n) - n;     // p(n, j) = row + j
    for (int k = (n >> 4) + lane; k < n_half; k += 32) {
        uint32_t w = __ldg(sample_bits + k);
        if (k == (n >> 4)) w &= 0xFFFFu << (n & 15);          // only j >= n
        while (w) {
            const int b = __ffs((int)w) - 1;
            w &= w - 1;
            const int j = 16 * k + b;
            atomicAdd(j == n ? cnt_f + n : x_f + row + j, 1);
        }
    }
}

// 16 bytes of the bit-field starting at byte `at` (zero beyond n_bytes), words assembled with static indices only
__device__ __forceinline__ uint4 load_flag_chunk(const uint8_t *__restrict__ flags, unsigned long long at, unsigned long long n_bytes)
{
    if (at + 16 <= n_bytes) return __ldg(reinterpret_cast<const uint4 *>(flags + at));
    uint32_t w[4] = {0, 0, 0, 0};
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int b = 0; b < 4; ++b)
            if (at + 4 * q + b < n_bytes) w[q] |= (uint32_t)flags[at + 4 * q + b] << (8 * b);
    return make_uint4(w[0], w[1], w[2], w[3]);
}

constexpr int kFlagUnroll = 4;   // 16-byte chunks per lane and iteration: 2 KiB of bit-field per warp in flight

// warp-stride over 2 KiB pieces of the bit-field; n_bytes = T * F * N / 8
__global__ void __launch_bounds__(256) flag_count_kernel(const uint8_t *__restrict__ flags, unsigned long long n_bytes, int n_inputs,
                                                          int n_freq, int32_t *__restrict__ x, int32_t *__restrict__ cnt)
{
    const int lane = threadIdx.x & 31;
    const unsigned long long warp = ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned long long n_warps = ((unsigned long long)gridDim.x * blockDim.x) >> 5;
    const unsigned long long n_chunks = (n_bytes + 15) >> 4;
    const unsigned long long n_pieces = (n_chunks + 32 * kFlagUnroll - 1) / (32 * kFlagUnroll);
    const long long n_pairs = (long long)n_inputs * (n_inputs + 1) / 2;
    const uint32_t sample_bytes = (uint32_t)n_inputs >> 3;
    for (unsigned long long piece = warp; piece < n_pieces; piece += n_warps) {
        uint4 v[kFlagUnroll];
        uint32_t any = 0;
#pragma unroll
        for (int u = 0; u < kFlagUnroll; ++u) {                // chunk index (piece * kFlagUnroll + u) * 32 + lane: coalesced 512 B per u
            v[u] = load_flag_chunk(flags, (((piece * kFlagUnroll + u) << 5) + lane) << 4, n_bytes);
            any |= v[u].x | v[u].y | v[u].z | v[u].w;
        }
        // "bit-field extraction is performed only if the 32-bit representation of the bit-field is non-zero"
        if (__ballot_sync(0xFFFFFFFFu, any != 0) == 0) continue;
        // the piece's first bit: sample s_first, input n_first, channel f_first (the only 64-bit divisions, once per piece)
        const unsigned long long bit_first = (piece * kFlagUnroll << 5) << 7;
        const unsigned long long s_first = bit_first / (unsigned)n_inputs;
        const uint32_t n_first = (uint32_t)(bit_first - s_first * (unsigned)n_inputs);
        const uint32_t f_first = (uint32_t)(s_first % (unsigned)n_freq);
#pragma unroll
        for (int u = 0; u < kFlagUnroll; ++u) {
            uint32_t nz = __ballot_sync(0xFFFFFFFFu, (v[u].x | v[u].y | v[u].z | v[u].w) != 0);
            while (nz) {                                       // lanes holding flags, one after the other, the whole warp helping
                const int src = __ffs((int)nz) - 1;
                nz &= nz - 1;
                const uint32_t chunk_rel = (uint32_t)(u << 5) + (uint32_t)src;     // 16-byte chunk inside the piece
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t mine = (q == 0) ? v[u].x : (q == 1) ? v[u].y : (q == 2) ? v[u].z : v[u].w;
                    uint32_t m = __shfl_sync(0xFFFFFFFFu, mine, src);
                    while (m) {                                // warp-uniform
                        const int b = __ffs((int)m) - 1;
                        m &= m - 1;
                        // sample and input of this bit, relative to the piece's first bit (32-bit arithmetic only)
                        const uint32_t rel = n_first + (chunk_rel << 7) + 32u * q + (uint32_t)b;
                        const uint32_t ds = rel / (uint32_t)n_inputs;
                        const int n = (int)(rel - ds * (uint32_t)n_inputs);
                        const int f = (int)((f_first + ds) % (uint32_t)n_freq);
                        flag_row_update_warp(reinterpret_cast<const uint16_t *>(flags + (s_first + ds) * sample_bytes), n_inputs, n,
                                             x + (size_t)f * n_pairs, cnt + (size_t)f * n_inputs, lane);
                    }
                }
            }
        }
    }
}

}  // namespace xc
