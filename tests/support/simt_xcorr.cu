// simt_xcorr.cu -- test support only: an on-device second opinion for whole-matrix comparisons at sizes where the CPU
// oracle takes minutes.  It is NOT part of libxcorr.so and shares nothing with it (no headers, no layout, no finalize
// pass): one thread per visibility, a plain integer loop over t on the definition
//     V_f[i,j] = sum_t x_i conj(x_j),  x = sext4(byte >> 4) + i sext4(byte & 15)        (BASELINE.json:north_star)
// written straight into the packed triangle int32[F][P][2], p(i,j) = i(2N-i+1)/2 + (j-i).
// Parity itself is always judged against oracle/; this kernel is held to the same oracle checks by the tests that use it.
#include <cstdint>
#include <cuda_runtime.h>

namespace {

constexpr int kTile = 16;    // inputs per tile side: one block = 16 x 16 visibilities
constexpr int kChunk = 64;   // time samples staged in shared memory at a time

__device__ __forceinline__ int sext4(int nibble) { return (nibble ^ 8) - 8; }

__global__ void __launch_bounds__(kTile * kTile) simt_xcorr_kernel(const uint8_t *__restrict__ frame, int n_inputs, int n_freq, int n_time,
                                                                   int32_t *__restrict__ out)
{
    const int bj = blockIdx.x, bi = blockIdx.y, f = blockIdx.z;
    if (bj < bi) return;
    __shared__ int8_t re_i[kChunk][kTile], im_i[kChunk][kTile], re_j[kChunk][kTile], im_j[kChunk][kTile];
    const int tj = threadIdx.x % kTile, ti = threadIdx.x / kTile;
    const int i = bi * kTile + ti, j = bj * kTile + tj;
    int32_t acc_re = 0, acc_im = 0;
    for (int t0 = 0; t0 < n_time; t0 += kChunk) {
        __syncthreads();
        for (int k = threadIdx.x; k < kChunk * kTile; k += kTile * kTile) {
            const int dt = k / kTile, n = k % kTile;
            const int t = t0 + dt;
            const int ni = bi * kTile + n, nj = bj * kTile + n;
            const int b_i = (t < n_time && ni < n_inputs) ? frame[((size_t)t * n_freq + f) * n_inputs + ni] : 0;
            const int b_j = (t < n_time && nj < n_inputs) ? frame[((size_t)t * n_freq + f) * n_inputs + nj] : 0;
            re_i[dt][n] = (int8_t)sext4(b_i >> 4); im_i[dt][n] = (int8_t)sext4(b_i & 15);
            re_j[dt][n] = (int8_t)sext4(b_j >> 4); im_j[dt][n] = (int8_t)sext4(b_j & 15);
        }
        __syncthreads();
#pragma unroll 8
        for (int dt = 0; dt < kChunk; ++dt) {
            const int hi = re_i[dt][ti], li = im_i[dt][ti], hj = re_j[dt][tj], lj = im_j[dt][tj];
            acc_re += hi * hj + li * lj;
            acc_im += li * hj - hi * lj;
        }
    }
    if (i <= j && j < n_inputs) {
        const long long n = n_inputs;
        const long long p = (long long)i * (2 * n - i + 1) / 2 + (j - i);
        const long long pairs = n * (n + 1) / 2;
        out[((long long)f * pairs + p) * 2 + 0] = acc_re;
        out[((long long)f * pairs + p) * 2 + 1] = acc_im;
    }
}

}  // namespace

// frame_dev: uint8[T][F][N]; out_dev: int32[F][P][2], fully overwritten.  Returns 0 or the cudaError_t.
extern "C" int simt_xcorr(const void *frame_dev, int n_inputs, int n_freq, int n_time, int32_t *out_dev, void *cuda_stream)
{
    if (!frame_dev || !out_dev || n_inputs <= 0 || n_freq <= 0 || n_freq > 65535 || n_time <= 0) return -1;
    const int nb = (n_inputs + kTile - 1) / kTile;
    if (nb > 65535) return -1;
    simt_xcorr_kernel<<<dim3(nb, nb, n_freq), kTile * kTile, 0, (cudaStream_t)cuda_stream>>>((const uint8_t *)frame_dev, n_inputs, n_freq,
                                                                                          n_time, out_dev);
    return (int)cudaGetLastError();
}
