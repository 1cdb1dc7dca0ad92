/*
 * xcorr_oracle.c -- CPU ORACLE for the X-engine correlation path.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is test infrastructure.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header,
 * table or helper with the CUDA path under paper_1503_06189_b200/ and neither imports the other.
 *
 * What it computes (the definition itself, not an approximation):
 *
 *   "the X-engine correlates all of the inputs against one another within each frequency band"
 *   (section I) and the kernels do "the actual cross-correlation and integration"
 *   (section II-B).  One sample is one byte, "a 4+4-bit complex number, so all 256
 *   inputs for one frequency take up 256 bytes"; a packet carries time samples x
 *   frequency bands x inputs with the input index fastest, i.e. frame[t][f][n].
 *
 *   The paper never prints the formula, nibble order, sign encoding or output order; those are the
 *   readings fixed in DESIGN.md section "Readings" (R1..R5, from BASELINE.json:north_star):
 *
 *     h(b) = sext4(b >> 4)   real part,      two's complement, range [-8, 7]      (R2, R3)
 *     l(b) = sext4(b & 15)   imaginary part
 *     Re V_f[i,j] = sum_t ( h_i*h_j + l_i*l_j )                                   (R1)
 *     Im V_f[i,j] = sum_t ( l_i*h_j - h_i*l_j )          i.e. V = sum_t x_i * conj(x_j)
 *     for 0 <= i <= j < N, written at out[f][p(i,j)][0..1], p(i,j) = i*(2N-i+1)/2 + (j-i)   (R4)
 *
 * Sums are exact integers: accumulated in int64, and every function returns nonzero if a value
 * does not fit the int32 output (R5) instead of wrapping.
 *
 * Two forms, both the plain definition:
 *   xcorr_oracle_naive   the literal loop nest (f, i<=j, t) on the packed bytes in place.
 *   xcorr_oracle_planar  first writes each channel's h and l as int8 arrays re[n][t], im[n][t]
 *                        (a change of storage order only), then the same loop nest with the t loop
 *                        contiguous; OpenMP over (f, i).  Must equal the naive form bit for bit
 *                        (tests/test_oracle_pins.py).  This one is the timed CPU baseline.
 *   xcorr_oracle_pairs   the naive inner loop for a caller-supplied list of (f, i, j) only, for
 *                        sampled checks at sizes where the full triangle takes minutes.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): hand-worked bytes, closed forms, one-hot/two-hot
 * indexing, Table I's 16,842,752-byte output size, numpy full N x N brute force,
 * Hermitian/sign symmetries, linearity over split frames, zero padding, Freivalds identities.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* R2/R3: 4-bit two's complement -> int.  0..7 stay, 8..15 map to -8..-1. */
static inline int sext4(unsigned v) { v &= 15u; return (int)v - (int)((v & 8u) << 1); }
static inline int re_of(uint8_t b) { return sext4((unsigned)b >> 4); }   /* high nibble */
static inline int im_of(uint8_t b) { return sext4((unsigned)b & 15u); }  /* low nibble  */

/* R4: row-major upper triangle including the diagonal. */
static inline int64_t pair_index(int64_t n_inputs, int64_t i, int64_t j)
{
    return i * (2 * n_inputs - i + 1) / 2 + (j - i);
}

int64_t xcorr_oracle_pair_index(int n_inputs, int i, int j) { return pair_index(n_inputs, i, j); }

int xcorr_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static inline int fits_i32(int64_t v) { return v >= INT32_MIN && v <= INT32_MAX; }

/* The literal definition.  frame: uint8[T][F][N].  out: int32[F][P][2].  Returns 0, or 1 on int32 overflow. */
int xcorr_oracle_naive(const uint8_t *frame, int n_inputs, int n_freq, int n_time, int32_t *out)
{
    const int64_t N = n_inputs, F = n_freq, T = n_time, P = N * (N + 1) / 2;
    int bad = 0;
    for (int64_t f = 0; f < F; ++f)
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = i; j < N; ++j) {
                int64_t re = 0, im = 0;
                for (int64_t t = 0; t < T; ++t) {
                    const uint8_t bi = frame[(t * F + f) * N + i];
                    const uint8_t bj = frame[(t * F + f) * N + j];
                    const int hi = re_of(bi), li = im_of(bi), hj = re_of(bj), lj = im_of(bj);
                    re += hi * hj + li * lj;
                    im += li * hj - hi * lj;
                }
                if (!fits_i32(re) || !fits_i32(im)) bad = 1;
                int32_t *o = out + (f * P + pair_index(N, i, j)) * 2;
                o[0] = (int32_t)re;
                o[1] = (int32_t)im;
            }
    return bad;
}

/* Same sums for listed (f,i,j) triples only.  idx: int32[n_pairs][3].  out: int64[n_pairs][2]. */
int xcorr_oracle_pairs(const uint8_t *frame, int n_inputs, int n_freq, int n_time,
                       const int32_t *idx, int64_t n_pairs, int64_t *out)
{
    const int64_t N = n_inputs, F = n_freq, T = n_time;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(| : bad)
    for (int64_t k = 0; k < n_pairs; ++k) {
        const int64_t f = idx[3 * k], i = idx[3 * k + 1], j = idx[3 * k + 2];
        if (f < 0 || f >= F || i < 0 || j < i || j >= N) { bad |= 2; continue; }
        int64_t re = 0, im = 0;
        for (int64_t t = 0; t < T; ++t) {
            const uint8_t bi = frame[(t * F + f) * N + i];
            const uint8_t bj = frame[(t * F + f) * N + j];
            const int hi = re_of(bi), li = im_of(bi), hj = re_of(bj), lj = im_of(bj);
            re += hi * hj + li * lj;
            im += li * hj - hi * lj;
        }
        out[2 * k] = re;
        out[2 * k + 1] = im;
    }
    return bad;
}

/*
 * Planar form.  Channels [f_begin, f_end) only (so a bounded sample of a big frame can be timed);
 * out is still indexed by absolute f, other channels are left untouched.
 * Returns 0, 1 on int32 overflow, 3 if scratch memory could not be allocated.
 */
int xcorr_oracle_planar_range(const uint8_t *frame, int n_inputs, int n_freq, int n_time,
                              int f_begin, int f_end, int32_t *out)
{
    const int64_t N = n_inputs, F = n_freq, T = n_time, P = N * (N + 1) / 2;
    int bad = 0;
    int8_t *re = (int8_t *)malloc((size_t)(N * T ? N * T : 1));
    int8_t *im = (int8_t *)malloc((size_t)(N * T ? N * T : 1));
    if (!re || !im) { free(re); free(im); return 3; }
    for (int64_t f = f_begin; f < f_end; ++f) {
        /* storage-order change only: re[n][t] = h(frame[t][f][n]), im[n][t] = l(frame[t][f][n]) */
#pragma omp parallel for schedule(static)
        for (int64_t t = 0; t < T; ++t)
            for (int64_t n = 0; n < N; ++n) {
                const uint8_t b = frame[(t * F + f) * N + n];
                re[n * T + t] = (int8_t)re_of(b);
                im[n * T + t] = (int8_t)im_of(b);
            }
#pragma omp parallel for schedule(dynamic, 1) reduction(| : bad)
        for (int64_t i = 0; i < N; ++i) {
            const int8_t *hi = re + i * T, *li = im + i * T;
            for (int64_t j = i; j < N; ++j) {
                const int8_t *hj = re + j * T, *lj = im + j * T;
                int64_t sre = 0, sim = 0;
                for (int64_t t = 0; t < T; ++t) {
                    sre += hi[t] * hj[t] + li[t] * lj[t];
                    sim += li[t] * hj[t] - hi[t] * lj[t];
                }
                if (!fits_i32(sre) || !fits_i32(sim)) bad |= 1;
                int32_t *o = out + (f * P + pair_index(N, i, j)) * 2;
                o[0] = (int32_t)sre;
                o[1] = (int32_t)sim;
            }
        }
    }
    free(re);
    free(im);
    return bad;
}

int xcorr_oracle_planar(const uint8_t *frame, int n_inputs, int n_freq, int n_time, int32_t *out)
{
    return xcorr_oracle_planar_range(frame, n_inputs, n_freq, n_time, 0, n_freq, out);
}
