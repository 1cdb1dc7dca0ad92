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
// only if the 32-bit representation of the bit-field is non-zero": the kernel reads 128 bits per
// thread and extracts bits only from non-zero words; the per-sample intersection work is O(E^2) as in the paper.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.hpp"

namespace xc {

// One flagged bit (sample s, input n): add 1 to X[f][p(n, j)] for every input j >= n flagged in the same sample
// (j == n gives the counter c_f[n] on the diagonal).  The sample's bit-field is n_inputs / 16 aligned halfwords.
__device__ __forceinline__ void flag_row_update(const uint16_t *__restrict__ sample_bits, int n_inputs, int n, int32_t *x_f)
{
    const int n_half = n_inputs >> 4;
    const long long row = pair_index(n_inputs, n, n) - n;     // p(n, j) = row + j
    for (int k = n >> 4; k < n_half; ++k) {
        uint32_t w = __ldg(sample_bits + k);
        if (k == (n >> 4)) w &= 0xFFFFu << (n & 15);          // only j >= n
        while (w) {
            const int b = __ffs((int)w) - 1;
            w &= w - 1;
            atomicAdd(x_f + row + (16 * k + b), 1);
        }
    }
}

// grid-stride over 16-byte chunks of the bit-field; n_bytes = T * F * N / 8
__global__ void __launch_bounds__(256) flag_count_kernel(const uint8_t *__restrict__ flags, unsigned long long n_bytes, int n_inputs,
                                                          int n_freq, int32_t *__restrict__ x)
{
    const unsigned long long n_chunks = (n_bytes + 15) >> 4;
    const long long n_pairs = (long long)n_inputs * (n_inputs + 1) / 2;
    const uint32_t sample_bytes = (uint32_t)n_inputs >> 3;
    for (unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; g < n_chunks;
         g += (unsigned long long)gridDim.x * blockDim.x) {
        uint32_t w[4] = {0, 0, 0, 0};
        if ((g << 4) + 16 <= n_bytes) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(flags) + g);
            w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
        } else {                                               // ragged last chunk
            for (unsigned long long b = g << 4; b < n_bytes; ++b) w[(b & 15) >> 2] |= (uint32_t)flags[b] << (8 * (b & 3));
        }
        if ((w[0] | w[1] | w[2] | w[3]) == 0) continue;        // the common case: nothing flagged in these 128 samples-bits
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t m = w[q];
            while (m) {
                const int b = __ffs((int)m) - 1;
                m &= m - 1;
                const unsigned long long bit = (g << 7) + 32u * q + b;     // global bit index = sample * N + input
                const unsigned long long s = bit / (unsigned)n_inputs;
                const int n = (int)(bit - s * (unsigned)n_inputs);
                const int f = (int)(s % (unsigned)n_freq);
                flag_row_update(reinterpret_cast<const uint16_t *>(flags + s * sample_bytes), n_inputs, n, x + (size_t)f * n_pairs);
            }
        }
    }
}

}  // namespace xc
