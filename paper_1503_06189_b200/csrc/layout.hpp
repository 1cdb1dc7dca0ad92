// layout.hpp -- shapes of the tiling and of the device accumulator (host + device).
//
// The visibility matrix of one channel is cut into SUPER-TILES of 256 x 256 inputs (one 2-CTA
// tcgen05 MMA, M = 256 = two CTAs x 128 TMEM lanes, N = 256).  Only super-tiles (I <= J) on or above
// the diagonal exist ("computes only upper-triangle tiles", BASELINE.json:north_star (b)).
//
// Device accumulator ("kernels add to the output of the last run").  A super-tile may be summed
// over time by several work segments (schedule.hpp); every segment owns one SLOT, so the epilogue needs no
// atomics between segments: it stores (first frame of an integration) or reduce-adds (later frames) into its own slot,
// and xcorr_read adds the slots of a tile together.  Slot layout -- TMEM-native:
//
//   acc[slot][r][row / 32][col / 4][row % 32][col % 4]   int32,   r in {0,1}, col in [0,512), row in [0,128)
//
// i.e. per epilogue warp (32 TMEM lanes) the columns run contiguously: a chunk of 32 columns is one 4 KiB piece, which
// the epilogue writes with eight 16-byte stores per lane (first frame: 512 contiguous bytes per warp and instruction) or
// stages in shared memory and hands to ONE bulk int32 reduce-add (later frames).
//
//     row          = TMEM lane       : input  i = 256*I + 128*r + row
//     col in [0,256)  "R" columns    : input  j = 256*J + col
//         I <  J :  value  Re V[i,j] = sum h_i h_j + l_i l_j
//         I == J :  value  G[i,j]    = sum (h_i + l_i)(h_j + l_j)
//     col in [256,512) "Q" columns   : input  j = 256*J + (col-256)
//         I <  J :  value  Im V[i,j] = sum l_i h_j - h_i l_j
//         I == J :  value  X[i,j]    = sum l_i h_j ;   Re V = G - X - X^T,  Im V = X - X^T  are formed by xcorr_read
//
// Lower-triangle R entries of diagonal super-tiles and anything with i >= N or j >= N are never read
// (and mostly never written).
//
// OFFSET OPERANDS.  The tensor core is fed x' = x + 8 in [0, 15] (h' = h + 8, l' = l + 8; and the complement
// 15 - l' where a negated operand is needed) instead of the sign-extended int8 value: the upper nibble of every
// operand byte is then constant zero, which measurably lowers the switching power of the MMA datapath (the part is
// power-limited).  The slots therefore hold the OFFSET sums
//     I <  J :  R'[i,j] = sum h'_i h'_j + l'_i l'_j          Q'[i,j] = sum l'_i h'_j + h'_i (15 - l'_j)
//     I == J :  R'[i,j] = sum (h'_i + l'_i)(h'_j + l'_j)      Q'[i,j] = sum l'_i h'_j
// and every segment also owns a row of per-input column sums over its time range ("sum slot"):
//
//   sums[slot][r][plane][row]   int32,  plane 0: sum_t h'   1: sum_t l'   of input 256*I + 128*r + row   (A block)
//                                       plane 2: sum_t h'   3: sum_t l'   of input 256*J + 128*r + row   (B block, I < J)
//
// xcorr_read removes the offsets exactly (finalize_kernel.cuh); all arithmetic is modulo 2^32 and the final values fit
// int32 by the overflow guard, so intermediate wrap-around of R', Q' is harmless (tcgen05 kind::i8 accumulators wrap).
#pragma once
#include <cstdint>

namespace xc {

constexpr int kBlock = 128;        // inputs per CTA row block (TMEM lanes)
constexpr int kSuper = 256;        // inputs per super-block (CTA pair)
constexpr int kAccCols = 512;      // TMEM columns per CTA: 256 R + 256 Q
constexpr int kDiagSplitCol = 192; // diagonal super-tiles: G[i < 128, j >= 192] is written by CTA half 1 (from its transposed copy) into half 0's place
constexpr int kAccElemsPerCta = kAccCols * kBlock;          // 65536 int32
constexpr int kAccElemsPerQuarter = kAccCols * 32;          // 16384 int32: the 32 TMEM lanes one epilogue warp owns
constexpr int kAccElemsPerSlot = 2 * kAccElemsPerCta;        // 131072 int32 = 512 KiB
constexpr int kSumPlanes = 4;                                // h'_A, l'_A, h'_B, l'_B
constexpr int kSumElemsPerCta = kSumPlanes * kBlock;          // 512 int32
constexpr int kSumElemsPerSlot = 2 * kSumElemsPerCta;         // 1024 int32 = 4 KiB

__host__ __device__ inline int n_super(int n_inputs) { return (n_inputs + kSuper - 1) / kSuper; }
__host__ __device__ inline int n_supertiles(int nb) { return nb * (nb + 1) / 2; }
// row-major upper triangle of super-blocks
__host__ __device__ inline int supertile_index(int nb, int I, int J) { return I * (2 * nb - I + 1) / 2 + (J - I); }
// R4: packed output pair index
__host__ __device__ inline long long pair_index(long long n, long long i, long long j) { return i * (2 * n - i + 1) / 2 + (j - i); }
// int32 offset of (r, col, row) inside a slot
__host__ __device__ inline size_t slot_offset(int r, int col, int row)
{
    return (size_t)r * kAccElemsPerCta + (size_t)(row >> 5) * kAccElemsPerQuarter + ((size_t)(col >> 2) * 32 + (row & 31)) * 4 + (col & 3);
}

}  // namespace xc
