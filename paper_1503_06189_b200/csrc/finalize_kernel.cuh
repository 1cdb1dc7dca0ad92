// finalize_kernel.cuh -- xcorr_read's kernel: accumulator slots (layout.hpp) -> packed upper triangle
// int32[F][P][2] (R4).
//
// A slot is [r][row/32][col/4][row%32][4] (layout.hpp), the output is row-major in (i, j).  Each block turns one
// 32 x 32 patch around through shared memory so that both sides are coalesced: 16-byte vector reads along the row
// index, 8-byte (re, im) writes along j.  The slots of a super-tile (one per work segment that summed part of
// its time range) are added here, and the operand offsets are removed (layout.hpp "OFFSET OPERANDS"): with
// h = h' - 8, l = l' - 8, the column sums sh_n = sum_t h'_n, sl_n = sum_t l'_n of the tile's sum slots and
// T' = the number of (zero-padded) samples the tensor path has integrated,
//
//   I < J (R' = sum h'_i h'_j + l'_i l'_j,  Q' = sum l'_i h'_j + h'_i (15 - l'_j)):
//     Re V[i,j] = R'[i,j] - 8 (sh_i + sl_i + sh_j + sl_j) + 128 T'
//     Im V[i,j] = Q'[i,j] - 7 sh_i - 8 sl_i - 8 sh_j + 8 sl_j
//   I == J (R' = G' = sum (h'_i + l'_i)(h'_j + l'_j),  Q' = X' = sum l'_i h'_j; xengine_kernel.cuh header):
//     G = G' - 16 (sh_i + sl_i + sh_j + sl_j) + 256 T',   X[i,j] = X'[i,j] - 8 sl_i - 8 sh_j + 64 T',   hence
//     Re V[i,j] = G - X[i,j] - X[j,i] = G'[i,j] - X'[i,j] - X'[j,i] - 8 (sh_i + sl_i + sh_j + sl_j) + 128 T'
//     Im V[i,j] = X[i,j] - X[j,i]     = X'[i,j] - X'[j,i] + 8 (sh_i - sl_i) - 8 (sh_j - sl_j)
//
// exactly, modulo 2^32 (unsigned arithmetic below; the true values fit int32 by the overflow guard).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.hpp"

namespace xc {

// sum over the tile's slots of the 4 consecutive columns [col4*4, col4*4+4) of row `row`, CTA half r
__device__ __forceinline__ uint4 slot_sum_v4(const int32_t *__restrict__ acc, int slot_begin, int slot_end, int r, int col4, int row)
{
    uint4 s = make_uint4(0, 0, 0, 0);
    for (int sl = slot_begin; sl < slot_end; ++sl) {
        // streaming (evict-first) load: a slot is dead once it has been read here
        const uint4 v = __ldcs(reinterpret_cast<const uint4 *>(acc + (size_t)sl * kAccElemsPerSlot + (size_t)r * kAccElemsPerCta +
                                                               (size_t)(row >> 5) * kAccElemsPerQuarter + ((size_t)col4 * 32 + (row & 31)) * 4));
        s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
    }
    return s;
}

// Lost-sample normalisation fused into the write (normalise_kernel.cuh): inputs of the kNormalise variant.
// The flag counters and the loss counters are double-buffered by integration: this read uses one half and, on its way, puts
// the OTHER half (read by the previous integration's finalize pass, which stream order has completed) back to zero -- so
// xcorr_read_normalized is this one kernel: no gather before it, no clearing pass after it.
struct NormParams {
    int32_t *x;              // device int32[F][P]: flag intersections (i < j); cleared here as they are read (each by exactly one thread)
    const int32_t *cnt;      // device int32[F][N]: flag counters c_f[n] of this integration
    int32_t *cnt_clear;      // device int32[F][N]: the other half, zeroed by the diagonal blocks
    const int32_t *lost;     // device int32[F]: time samples lost with their packets, per channel, this integration
    int32_t *lost_clear;     // device int32[F]: the other half, zeroed by block (0, 0, f)
    int32_t *lost_out;       // device int32[F][P] or nullptr: the normalisation matrix L itself
    uint32_t n_samples;      // T: samples integrated since the last read
};

// grid (nt, nt, F), nt = ceil(N / 32); block 256 threads.  kNormalise = false: out = int32[F][P][2] (xcorr_read);
// kNormalise = true: out = float32[F][P][2] = V * T / (T - L) (xcorr_read_normalized)
template <bool kNormalise>
__global__ void __launch_bounds__(256) finalize_kernel(const int32_t *__restrict__ acc, const int32_t *__restrict__ sums,
                                                        const int32_t *__restrict__ tile_slot_begin, void *__restrict__ out_v, int n_inputs,
                                                        uint32_t offset_samples, const NormParams np)
{
    int32_t *__restrict__ out = reinterpret_cast<int32_t *>(out_v);
    const int bj = blockIdx.x, bi = blockIdx.y, f = blockIdx.z;
    // PDL (griddepcontrol): let the next kernel of the stream start its prologue; wait for the producer of the slots
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (bj < bi) return;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    __shared__ uint32_t sR[32][33];   // [col][row]
    __shared__ uint32_t sQ[32][33];   // [col][row]
    __shared__ uint32_t sX[32][33];   // [row j][col i] of the transposed patch (diagonal super-tiles only)
    __shared__ uint32_t sS[4][32];    // column sums: [0] sh_i [1] sl_i (rows of the patch)  [2] sh_j [3] sl_j (columns)
    __shared__ int32_t sC[2][32];     // kNormalise: flag counters c_f[i] of the patch's rows [0] and columns [1]
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // ty in 0..7
    const int nb = n_super(n_inputs), nst = n_supertiles(nb);
    const int i0 = bi * 32, j0 = bj * 32;
    const int I = i0 / kSuper, J = j0 / kSuper;
    const bool diag_super = (I == J);
    const int tile = f * nst + supertile_index(nb, I, J);
    const int sb = tile_slot_begin[tile], se = tile_slot_begin[tile + 1];

    // kNormalise: the flag intersections X_ij of the four pairs this thread writes in phase 2 (rows i0 + ty + 8k, column j0 + tx:
    // 128 B contiguous per warp and row) are fetched here, with the slot loads, so phase 2 has no second round of loads
    int32_t x_pre[4] = {0, 0, 0, 0};
    if constexpr (kNormalise) {
        const long long PP = (long long)n_inputs * (n_inputs + 1) / 2;
        const int j = j0 + tx;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int i = i0 + ty + 8 * k;
            if (j < n_inputs && i < j) x_pre[k] = np.x[(long long)f * PP + pair_index(n_inputs, i, j)];
        }
    }
    // phase 1: thread (tx = row, ty = group of 4 columns): 16-byte loads, 512 B contiguous per warp
    {
        const int il = (i0 % kSuper) + tx;            // row inside the super-block
        const int r = il / kBlock, row = il % kBlock;
        const int c4 = ((j0 % kSuper) >> 2) + ty;     // column group inside the super-block
        const uint4 vr = slot_sum_v4(acc, sb, se, r, c4, row);
        const uint4 vq = slot_sum_v4(acc, sb, se, r, 64 + c4, row);
        sR[4 * ty + 0][tx] = vr.x; sR[4 * ty + 1][tx] = vr.y; sR[4 * ty + 2][tx] = vr.z; sR[4 * ty + 3][tx] = vr.w;
        sQ[4 * ty + 0][tx] = vq.x; sQ[4 * ty + 1][tx] = vq.y; sQ[4 * ty + 2][tx] = vq.z; sQ[4 * ty + 3][tx] = vq.w;
        if (diag_super) {
            // X[j][i] for rows j in [j0, j0+32), columns i in [i0, i0+32)
            const int jl = (j0 % kSuper) + tx;
            const uint4 vx = slot_sum_v4(acc, sb, se, jl / kBlock, 64 + ((i0 % kSuper) >> 2) + ty, jl % kBlock);
            sX[tx][4 * ty + 0] = vx.x; sX[tx][4 * ty + 1] = vx.y; sX[tx][4 * ty + 2] = vx.z; sX[tx][4 * ty + 3] = vx.w;
        }
        if constexpr (kNormalise) {
            // the counters of the patch's rows and columns: two coalesced 128-byte loads per block, beside the slot loads
            if (ty >= 4 && ty < 6) {
                const int nn = ((ty == 4) ? i0 : j0) + tx;
                sC[ty - 4][tx] = (nn < n_inputs) ? np.cnt[(size_t)f * n_inputs + nn] : 0;
            }
            // the other half of the double-buffered counters goes back to zero (see NormParams)
            if (bi == bj && ty == 6 && i0 + tx < n_inputs) np.cnt_clear[(size_t)f * n_inputs + i0 + tx] = 0;
            if (bi == 0 && bj == 0 && threadIdx.x == 255) np.lost_clear[f] = 0;
        }
        if (ty < 4) {
            // ty 0,1: sh, sl of row input i0 + tx (A block of its CTA half); ty 2,3: of column input j0 + tx
            // (A block again on a diagonal super-tile, the B block for I < J)
            const int nl = ((ty < 2) ? (i0 % kSuper) : (j0 % kSuper)) + tx;
            const int plane = (ty & 1) + ((ty >= 2 && !diag_super) ? 2 : 0);
            uint32_t v = 0;
            for (int sl = sb; sl < se; ++sl)
                v += (uint32_t)sums[(size_t)sl * kSumElemsPerSlot + (size_t)(nl / kBlock) * kSumElemsPerCta + plane * kBlock + (nl % kBlock)];
            sS[ty][tx] = v;
        }
    }
    __syncthreads();
    // phase 2: tx <-> column j0 + tx, one output row per ty step: 8-byte (re, im) writes, 256 B contiguous per warp
    const long long P = (long long)n_inputs * (n_inputs + 1) / 2;
    const uint32_t shj = sS[2][tx], slj = sS[3][tx];
    int32_t x_jj = 0, lost_f = 0;
    float scale_f = 0.0f;             // the scale of a pair neither of whose inputs was ever flagged: the packet loss alone
    if constexpr (kNormalise) {
        x_jj = sC[1][tx];
        lost_f = np.lost[f];
        const int32_t valid_f = (int32_t)np.n_samples - lost_f;
        scale_f = (valid_f > 0) ? __fdiv_rn((float)np.n_samples, (float)valid_f) : 0.0f;
    }
#pragma unroll(kNormalise ? 4 : 1)
    for (int k = 0; k < 4; ++k) {
        const int ic = ty + 8 * k;
        const int i = i0 + ic, j = j0 + tx;
        if (j < n_inputs && i <= j) {
            const uint32_t shi = sS[0][ic], sli = sS[1][ic];
            uint32_t re = sR[tx][ic] - 8u * (shi + sli + shj + slj) + 128u * offset_samples;
            uint32_t im;
            if (diag_super) {
                re -= sQ[tx][ic] + sX[tx][ic];
                im = (i == j) ? 0u : sQ[tx][ic] - sX[tx][ic] + 8u * (shi - sli) - 8u * (shj - slj);
            } else {
                im = sQ[tx][ic] - 7u * shi - 8u * sli - 8u * shj + 8u * slj;
            }
            const long long p = (long long)f * P + pair_index(n_inputs, i, j);
            if constexpr (kNormalise) {
                // L = lost + c_i + c_j - X_ij (the point (i, i) receives its counter once); V~ = V * T / (T - L)
                const int32_t x_ii = sC[0][ic];
                const int32_t x_ij = x_pre[k];
                if (x_ij) np.x[p] = 0;                 // ends the integration: this thread is the only reader of X[p]
                const int32_t lost_ij = lost_f + x_ii + ((i != j) ? (x_jj - x_ij) : 0);
                float scale = scale_f;
                if (lost_ij != lost_f) {               // same expression, evaluated only where a flag counter comes in
                    const int32_t valid = (int32_t)np.n_samples - lost_ij;
                    scale = (valid > 0) ? __fdiv_rn((float)np.n_samples, (float)valid) : 0.0f;
                }
                __stcs(reinterpret_cast<float2 *>(reinterpret_cast<float *>(out_v) + p * 2),
                       make_float2(__fmul_rn((float)(int32_t)re, scale), __fmul_rn((float)(int32_t)im, scale)));
                if (np.lost_out) np.lost_out[p] = lost_ij;
            } else {
                __stcs(reinterpret_cast<int2 *>(out + p * 2), make_int2((int32_t)re, (int32_t)im));
            }
        }
    }
}

}  // namespace xc
