// finalize_kernel.cuh -- xcorr_read's kernel: device accumulator (layout.hpp) -> packed upper triangle
// int32[F][P][2] (R4), and the SIMT cross-check kernel used only by the tests.
//
// The accumulator is column-major per CTA tile (row = TMEM lane is the fast index), the output is row-major
// in (i, j); each block turns one 32 x 32 patch around through shared memory so that both sides are
// 128-byte coalesced.  On diagonal super-tiles Im V[i,j] = X[i,j] - X[j,i] (layout.hpp).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.hpp"

namespace xc {

__device__ __forceinline__ const int32_t *acc_elem(const int32_t *acc, int nst, int nb, int f, int i, int j, int q_cols)
{
    // element for row input i, column input j (i's super-block <= j's); q_cols = 0 -> R, 256 -> Q
    const int I = i / kSuper, J = j / kSuper;
    const int tile = f * nst + supertile_index(nb, I, J);
    const int r = (i % kSuper) / kBlock;
    return acc + ((size_t)tile * 2 + r) * (size_t)kAccElemsPerCta + (size_t)(q_cols + j % kSuper) * kBlock + (i % kBlock);
}

// grid (nt, nt, F), nt = ceil(N / 32); block (32, 8)
__global__ void __launch_bounds__(256) finalize_kernel(const int32_t *__restrict__ acc, int32_t *__restrict__ out, int n_inputs)
{
    const int bj = blockIdx.x, bi = blockIdx.y, f = blockIdx.z;
    if (bj < bi) return;
    __shared__ int32_t sR[32][33];
    __shared__ int32_t sQ[32][33];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int nb = n_super(n_inputs), nst = n_supertiles(nb);
    const int i0 = bi * 32, j0 = bj * 32;
    const bool diag_super = (i0 / kSuper) == (j0 / kSuper);

    // phase 1: coalesced reads along the row index (tx <-> row i0 + tx), one column per ty step
    for (int cc = ty; cc < 32; cc += 8) {
        const int i = i0 + tx, j = j0 + cc;
        int32_t r = 0, q = 0;
        if (i < n_inputs && j < n_inputs) {
            r = *acc_elem(acc, nst, nb, f, i, j, 0);
            q = *acc_elem(acc, nst, nb, f, i, j, 256);
        }
        sR[cc][tx] = r;
        sQ[cc][tx] = q;
    }
    __syncthreads();
    // phase 2: tx <-> column j0 + tx, one output row per ty step; X[j,i] is read coalesced along j
    const long long P = (long long)n_inputs * (n_inputs + 1) / 2;
    for (int ic = ty; ic < 32; ic += 8) {
        const int i = i0 + ic, j = j0 + tx;
        if (i < n_inputs && j < n_inputs && i <= j) {
            int32_t re = sR[tx][ic];
            int32_t im = sQ[tx][ic];
            if (diag_super) im = (i == j) ? 0 : im - *acc_elem(acc, nst, nb, f, j, i, 256);
            int2 v = make_int2(re, im);
            *reinterpret_cast<int2 *>(out + ((long long)f * P + pair_index(n_inputs, i, j)) * 2) = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// SIMT cross-check ("second opinion" for the GPU tests at sizes where the CPU oracle takes minutes).
// One thread per accumulator element, plain integer loop over t.  NOT used by xcorr_process.
// grid: n_tiles * 2 * (128 / 8) blocks, block 256 threads (thread <-> column), 8 rows per block.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) simt_reference_kernel(const uint8_t *__restrict__ frame, int32_t *acc, int n_inputs, int n_freq,
                                                             int n_time)
{
    constexpr int kRows = 8;
    const int nb = n_super(n_inputs), nst = n_supertiles(nb);
    int b = blockIdx.x;
    const int rowgrp = b % (kBlock / kRows); b /= (kBlock / kRows);
    const int r = b % 2; b /= 2;
    const int tile = b;
    const int f = tile / nst;
    int st = tile % nst, I = 0;
    while (st >= nb - I) { st -= nb - I; ++I; }
    const int J = I + st;
    const int col = threadIdx.x;
    const int j = J * kSuper + col;
    const bool diag = (I == J);
    int32_t accR[kRows], accQ[kRows];
#pragma unroll
    for (int k = 0; k < kRows; ++k) accR[k] = accQ[k] = 0;
    const int row_base = rowgrp * kRows;
    const int i_base = I * kSuper + r * kBlock + row_base;
    for (int t = 0; t < n_time; ++t) {
        const uint8_t *line = frame + ((size_t)t * n_freq + f) * n_inputs;
        const int bjv = (j < n_inputs) ? line[j] : 0;
        const int hj = (int)(int8_t)(bjv & 0xF0) >> 4, lj = (int)(int8_t)((bjv & 15) << 4) >> 4;
#pragma unroll
        for (int k = 0; k < kRows; ++k) {
            const int i = i_base + k;
            const int biv = (i < n_inputs) ? line[i] : 0;
            const int hi = (int)(int8_t)(biv & 0xF0) >> 4, li = (int)(int8_t)((biv & 15) << 4) >> 4;
            accR[k] += hi * hj + li * lj;
            accQ[k] += diag ? li * hj : li * hj - hi * lj;
        }
    }
    int32_t *base = acc + ((size_t)tile * 2 + r) * (size_t)kAccElemsPerCta;
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
        atomicAdd(base + (size_t)col * kBlock + row_base + k, accR[k]);
        atomicAdd(base + (size_t)(256 + col) * kBlock + row_base + k, accQ[k]);
    }
}

}  // namespace xc
