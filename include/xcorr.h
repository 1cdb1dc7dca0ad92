/*
 * xcorr.h -- C ABI of the B200 X-engine correlation library (libxcorr.so).
 *
 * The library computes, on ONE NVIDIA B200 (compute capability 10.0, sm_100a), the data-parallel hot
 * path of the CHIME Pathfinder X-engine (arxiv 1503.06189):
 *
 *   "the X-engine correlates all of the inputs against one another within each frequency band"
 *                                                                   (section I)
 *   "A set of GPU programs called kernels do the actual cross-correlation and integration."
 *                                                                   (section II-B)
 *   "the correlation kernels simply add to the output of the last run, extending the integration
 *    time of the output"; the copy back to the host "is not run on every invocation"
 *                                                                   (section II-B)
 *
 * For every frequency channel f and every input pair 0 <= i <= j < N it accumulates, over all time
 * samples handed to xcorr_process() since the last xcorr_read(),
 *
 *     V_f[i,j] = sum_t x_f,t[i] * conj(x_f,t[j])          (BASELINE.json:north_star; R1)
 *
 * as exact int32 real / imaginary sums.  One sample is one byte, a 4+4-bit complex number
 * (PAPER.md:29, :67): real part in the high nibble, imaginary part in the low nibble, each signed
 * 4-bit two's complement in [-8, 7] (R2, R3).  The value -8 is legal.
 *
 * Conventions
 *   - Every function returns XCORR_OK (0) or a negative XCORR_E* code; nothing aborts or throws.
 *   - "dev" pointers are CUDA device pointers on the device that was current at xcorr_create();
 *     "host" pointers are ordinary (preferably page-locked) host pointers.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - A handle is not thread safe; use it from one host thread at a time, with the device it was created on current
 *     (a call made while another device is current returns XCORR_EINVAL).
 *   - Stream order.  The device state of a handle (accumulator, flag / loss accumulators) is ordered by the streams the
 *     calls are given: calls on the SAME stream run in stream order; a call given ANOTHER stream than the handle's
 *     previous call first makes that stream wait, on the device (cudaStreamWaitEvent), for everything enqueued so far
 *     on the previous stream -- so xcorr_process on stream A followed by xcorr_read on stream B is safe and exact.  A
 *     stream handed to a call must therefore stay alive until the handle's next call has returned (or the handle is
 *     destroyed).  Destroying it earlier is undefined behaviour, as for any CUDA call on a dead stream: the next call
 *     records an event on it.  Where CUDA happens to report the stream as invalid the call returns XCORR_EINVAL, but
 *     that is a courtesy, not a contract.  (The Python wrappers keep the last stream object referenced for this reason.)
 *     The host-side bookkeeping (first frame of an integration, overflow guard, sample count) follows the order of the
 *     CALLS.
 *   - Nothing is allocated or freed after xcorr_create()/xcorr_stream_create() return (PAPER.md:49:
 *     "the entire application does not malloc or free any memory outside of startup and shutdown").
 *   - There is no CPU fallback: on a machine without an sm_100 GPU xcorr_create() fails with
 *     XCORR_EARCH / XCORR_ECUDA.
 */
#ifndef XCORR_H_
#define XCORR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define XCORR_OK          0
#define XCORR_EINVAL     -1   /* bad argument (NULL, non-positive size, N % 16 != 0, misaligned pointer, size overflow) */
#define XCORR_EARCH      -2   /* current device is not compute capability 10.x */
#define XCORR_ENOMEM     -3   /* device or host allocation failed */
#define XCORR_ECUDA      -4   /* a CUDA runtime/driver call failed; xcorr_last_cuda_error() has the code */
#define XCORR_EOVERFLOW  -5   /* this frame could push an int32 sum past 2^31-1; nothing was launched */
#define XCORR_ELIMIT     -6   /* larger than a built-in, never-allocated scratch table (xcorr_assemble_static); nothing was launched */

typedef struct xcorr_handle xcorr_handle;
typedef struct xcorr_stream xcorr_stream;

/*
 * xcorr_create -- fix the problem shape and allocate everything (shapes are fixed at
 * startup in the paper's system too).
 *
 *   n_inputs     N  > 0, a multiple of 16 (TMA needs 16-byte global strides; the paper's N are 16, 256, 2048)
 *   n_freq       F  > 0 frequency channels per frame
 *   t_per_frame  T  > 0 time samples per frame (any value; the tail of the last tile is zero-filled,
 *                   which is exact because a zero sample adds nothing)
 *   out          receives the handle, owned by the library until xcorr_destroy()
 *
 * Allocates the device accumulator (zeroed), the work schedule and a device staging buffer of
 * xcorr_output_bytes() for host reads.  Errors: EINVAL, EARCH, ENOMEM, ECUDA.
 */
int xcorr_create(int n_inputs, int n_freq, int t_per_frame, xcorr_handle **out);

/*
 * xcorr_process -- correlate one frame and ADD it into the running integration.
 *
 *   packed_frame_dev  device pointer, exactly N*F*T bytes, layout uint8[t][f][input] with the input
 *                     index fastest (the packet payload "can be used by the GPU without
 *                     modification"); must be 16-byte aligned.  BORROWED: the caller keeps it alive
 *                     and unmodified until `cuda_stream` has passed this call.
 *   cuda_stream       the work is enqueued on this stream; the call does not synchronise.
 *
 * Steps run on the GPU (DESIGN.md section "Kernels"): TMA staging of 128-byte rows (a1), nibble unpack
 * to int8 planes (a2), tcgen05 kind::i8 Hermitian rank-T update with int32 accumulators in TMEM (a3),
 * epilogue add into the device accumulator (a4).
 * Errors: EINVAL (NULL / misaligned), EOVERFLOW if 128*(samples since last read + T) > 2^31-1
 * (checked on the host before anything is launched), ECUDA.
 */
int xcorr_process(xcorr_handle *h, const void *packed_frame_dev, void *cuda_stream);

/*
 * xcorr_promise_complete_frames -- optional promise about the frames handed to xcorr_process() on this handle.
 *
 * xengine_kernel is launched with programmatic dependent launch, so it may begin while the previous kernel of the
 * stream is still finishing.  By default its first frame load therefore waits for that kernel, in case it is the
 * producer of the frame and signalled launch completion early.  With `enabled` != 0 the caller promises that a frame
 * is never the output of a kernel that signals programmatic launch completion (cudaTriggerProgrammaticLaunchCompletion /
 * griddepcontrol.launch_dependents) before it has finished writing it.  Frames that are resident, that arrive by
 * cudaMemcpy, or that are written by ordinary kernels or by this library's assemble_kernel all qualify.  The frame is then
 * loaded, unpacked and multiplied while the previous xcorr_read / xcorr_process of the stream drains (C2: about 2 us per
 * frame); the accumulator is still guarded (the epilogue waits for the previous kernel before it touches a slot).
 * Errors: EINVAL (NULL handle).
 */
int xcorr_promise_complete_frames(xcorr_handle *h, int enabled);

/*
 * xcorr_read -- end the integration: write the visibilities and clear the accumulator (PAPER.md:99:
 * the device-to-host copy happens only at the end of an integration).
 *
 *   upper_triangle_out  int32[F][P][2], P = N(N+1)/2, pair index p(i,j) = i(2N-i+1)/2 + (j-i) for
 *                       i <= j (row-major upper triangle including the autocorrelations, R4;
 *                       size pinned by Table I), [0] = Re, [1] = Im.
 *                       May be a device pointer (stream-ordered; returns without synchronising) or a
 *                       host pointer (the call returns after the data has landed).  Caller-owned,
 *                       xcorr_output_bytes() bytes, 16-byte aligned if on the device.
 *   cuda_stream         stream to order the read on (after the xcorr_process calls it should include).
 *
 * The read ends the integration: the next xcorr_process starts from zero (its epilogue overwrites the accumulator slots
 * instead of adding to them -- there is no clearing pass), a second xcorr_read without a frame in between returns zeros,
 * and the sample counter used for the overflow guard is reset.
 * Errors: EINVAL, ECUDA.
 */
int xcorr_read(xcorr_handle *h, int32_t *upper_triangle_out, void *cuda_stream);

/* ---------------------------------------------------------------------------------------------------
 * Lost-sample normalisation (SURVEY.md 8(f) NEXT-1; section II-C, :111-121).  Samples lost to packet
 * loss or flagged by the F-engine are ZERO in the frame ("the data points are zeroed, before they are
 * transferred to the GPU", :113), so some visibilities hold fewer samples.  The paper's post-processing builds a
 * normalisation matrix -- a packet-loss counter added to every point (:115), per-(input, frequency) flag
 * counters (:116), minus the per-sample intersections of inputs flagged together (:117-119) -- and applies the
 * lost fraction to the correlation matrix (:121).  Readings N1..N5 in DESIGN.md section 12.
 * ------------------------------------------------------------------------------------------------- */

/*
 * xcorr_norm_enable -- startup-time call (no allocation after startup): allocates the device
 * flag-intersection accumulator int32[F][P] (zeroed), the packet-loss counters and the staging for host
 * reads of the normalisation matrix.  Idempotent.  Must not be called in the middle of an integration.
 * Errors: EINVAL, ENOMEM, ECUDA.
 */
int xcorr_norm_enable(xcorr_handle *h);

/*
 * xcorr_norm_process -- account for the lost samples of ONE frame (the frame given to xcorr_process before or
 * after this call, in the same integration).  Either pointer may be NULL.
 *
 *   flags_dev          device pointer, F-engine flag bit-field of the frame, uint8[T][F][N/8]: input n of sample
 *                      (t, f) is bit (n % 8) of byte n / 8; a set bit means that sample's voltage byte is zero in
 *                      the frame.  16-byte aligned, BORROWED until `cuda_stream` has passed this call.  One launch
 *                      of flag_count_kernel adds the per-sample intersections (and, on the diagonal, the flag
 *                      counters) into the handle's accumulator.
 *   lost_samples_host  HOST pointer, int32[F]: time samples of each channel lost with their packets in this
 *                      frame (0 <= value <= T; the paper's packet-loss counter, kept per channel: a stream's
 *                      counter applies to its 8 channels).  Read before the call returns.
 * Errors: EINVAL (normalisation not enabled, misaligned, counter out of range), ECUDA.  A call that fails has counted
 * nothing (neither flags nor lost samples), so it can be repeated as a whole.
 */
int xcorr_norm_process(xcorr_handle *h, const uint8_t *flags_dev, const int32_t *lost_samples_host, void *cuda_stream);

/*
 * xcorr_read_normalized -- xcorr_read() with the lost fraction applied, fused into the same kernel:
 *
 *   L[f][p(i,j)]  = lost[f] + c_f[i] + c_f[j] - #{samples with i and j both flagged}   (i != j)
 *   L[f][p(i,i)]  = lost[f] + c_f[i]
 *   vis_out       float32[F][P][2] = V * T / (T - L), T = samples integrated since the last read, computed in
 *                 float32 (int32 -> float, one division, one multiplication, each rounded to nearest); 0 where
 *                 T - L <= 0.  Pair order, host/device pointer rules and alignment as in xcorr_read.
 *   lost_matrix_out  optional (NULL to skip): int32[F][P], the normalisation matrix L itself (exact).
 *
 * Ends the integration: visibilities, flag accumulator and loss counters start again from zero (a plain
 * xcorr_read on a handle with normalisation enabled clears them as well).
 * Errors: EINVAL, ECUDA.
 */
int xcorr_read_normalized(xcorr_handle *h, float *vis_out, int32_t *lost_matrix_out, void *cuda_stream);

/* Release everything the handle owns (synchronises the device first).  NULL is a no-op. */
void xcorr_destroy(xcorr_handle *h);

/* Static, never-NULL description of an XCORR_* code. */
const char *xcorr_strerror(int code);

/* cudaError_t of the most recent failing CUDA call made through this handle (0 if none). */
int xcorr_last_cuda_error(const xcorr_handle *h);

/* N*F*T: bytes xcorr_process() reads.  F*P*8: bytes xcorr_read() writes.  0 for a NULL handle. */
size_t xcorr_frame_bytes(const xcorr_handle *h);
size_t xcorr_output_bytes(const xcorr_handle *h);

/* Total number of this library's kernels launched through the handle so far (bench.py's gpu_launches). */
uint64_t xcorr_kernel_launches(const xcorr_handle *h);

/* ---------------------------------------------------------------------------------------------------
 * Streamed frame path (hot-path row a5; stands in for the paper's ring buffers, and the
 * copy/compute pipeline of Fig. 4): page-locked host frames are copied to one of
 * `depth` device frame buffers on a copy stream while earlier frames are correlated on a compute
 * stream; CUDA events order the two.  "large (32 MB or greater) frames transferred most efficiently ...
 * page-locked".
 * ------------------------------------------------------------------------------------------------- */

/*
 * xcorr_stream_create -- allocate `depth` (>= 2, <= 8) device frame buffers of xcorr_frame_bytes(),
 * two CUDA streams and the events.  The xcorr_stream borrows `h` (destroy the stream first).
 * Errors: EINVAL, ENOMEM, ECUDA.
 */
int xcorr_stream_create(xcorr_handle *h, int depth, xcorr_stream **out);

/*
 * xcorr_stream_submit -- enqueue one host frame: H2D copy into the next device buffer, then xcorr_process on the
 * compute stream.  Ring back-pressure: if the correlation that last used that device buffer has not finished, the call
 * blocks the HOST thread until it has (cudaEventSynchronize).
 * `frame_host` (N*F*T bytes, layout as above) should be page-locked (cudaHostAlloc / cudaHostRegister /
 * torch pin_memory) for the copy to overlap; BORROWED until the matching copy has completed, i.e. until
 * `depth` further submits have returned or xcorr_stream_sync()/xcorr_stream_read() returns.
 * Returns without waiting for the GPU unless all `depth` buffers are still in flight.
 * Errors: EINVAL, EOVERFLOW, ECUDA.
 */
int xcorr_stream_submit(xcorr_stream *s, const void *frame_host);

/* Block until every submitted frame has been copied and correlated. */
int xcorr_stream_sync(xcorr_stream *s);

/*
 * xcorr_stream_read -- xcorr_read() ordered after all submitted frames on the compute stream.
 * `upper_triangle_out` host or device as in xcorr_read; returns after the data has landed.
 */
int xcorr_stream_read(xcorr_stream *s, int32_t *upper_triangle_out);

/*
 * xcorr_stream_read_async -- the same read enqueued on the compute stream WITHOUT waiting: the call returns at once,
 * the next xcorr_stream_submit() may follow immediately (its host-to-device copy then overlaps this read's kernel
 * and device-to-host copy -- PCIe is full duplex), and `upper_triangle_out` (host, page-locked for the overlap, or
 * device) holds the result once xcorr_stream_sync() has returned.  BORROWED until then.  Ends the integration like
 * xcorr_read(): frames submitted afterwards belong to the next one.
 */
int xcorr_stream_read_async(xcorr_stream *s, int32_t *upper_triangle_out);

/* Release buffers, streams and events (synchronises first).  NULL is a no-op. */
void xcorr_stream_destroy(xcorr_stream *s);

#ifdef __cplusplus
}
#endif
#endif /* XCORR_H_ */
