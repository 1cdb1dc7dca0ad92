/*
 * xcorr_assemble.h -- C ABI of the packet -> frame assembly stage (libxcorr.so).
 *
 * What the paper's network threads do on the CPU (section II-A, :59-:81) as GPU kernels, directly
 * upstream of xcorr_process():
 *
 *   "All that is required of the system is to place that data into the right location in a large host frame"
 *
 *   "all 256 inputs for one frequency take up 256 bytes.  For 8 frequency bands this represents 2KB. ... 4 time
 *    samples are recorded in each packet.  The header contains a streamID that identifies which frequency bands
 *    are represented in the packet, and a sequence number which gives the relative time"
 *   "When the system detects packet loss, it writes zeros into the area of the GPU staging buffer where the
 *    missing packet would have been placed. ... In the case of out of order packets, the sequence number is used
 *    to copy the packet into the correct location.  Duplicate packets are simply ignored."
 *   "The network threads track packet loss and F-engine error flags", the flags being
 *   "bit-fields in the packet footers".
 *
 * Wire format of one packet (reading P1; Fig. 3 of the paper did not survive), little endian:
 *
 *     offset 0   u32 magic      = XCORR_PACKET_MAGIC
 *            4   u32 stream_id    carries channels [C*stream_id, C*stream_id + C)
 *            8   u64 seq          array-wide index of the packet's FIRST time sample (P2)
 *           16   16 reserved bytes
 *           32   payload uint8[S][C][N]      (input fastest: usable by the GPU unmodified)
 *     32+S*C*N   footer  uint8[S][C][N/8]    flag bits, input n = bit (n % 8) of byte n / 8 (N1)
 *
 * S = samples per packet (4 in the paper), C = channels per stream (8), N = inputs (256): 9248 bytes ("~9K", :59).
 * Packets lie back to back in ARRIVAL order in one buffer, packet k at byte k * xcorr_assembler_packet_bytes().
 *
 * Conventions as in xcorr.h: int return codes (XCORR_OK or a negative XCORR_E*), nothing allocated after create,
 * no CPU fallback.
 */
#ifndef XCORR_ASSEMBLE_H_
#define XCORR_ASSEMBLE_H_

#include <stddef.h>
#include <stdint.h>

#include "xcorr.h"

#ifdef __cplusplus
extern "C" {
#endif

#define XCORR_PACKET_MAGIC        0x58454E47u
#define XCORR_PACKET_HEADER_BYTES 32

typedef struct xcorr_assembler xcorr_assembler;

/*
 * xcorr_assembler_create -- fix the shapes and allocate the position-ownership table and counters.
 *
 *   n_inputs, n_freq, t_per_frame   the frame shape uint8[T][F][N] of the xcorr handle this feeds
 *   samples_per_packet  S > 0, T % S == 0
 *   freq_per_packet     C > 0, F % C == 0, and C * N a multiple of 128 (rows of the payload and of the footer are
 *                       then whole 16-byte vectors; true for the paper's C = 8 and any legal N)
 * Errors: EINVAL, EARCH, ENOMEM, ECUDA.
 */
int xcorr_assembler_create(int n_inputs, int n_freq, int t_per_frame, int samples_per_packet, int freq_per_packet,
                           xcorr_assembler **out);

/* 32 + S*C*N + S*C*N/8.  0 for NULL. */
size_t xcorr_assembler_packet_bytes(const xcorr_assembler *a);

/*
 * xcorr_assemble -- build ONE frame from the packets that arrived for it.  Asynchronous on `cuda_stream`.
 *
 *   packets     n_packets packets back to back in arrival order.  Any pointer the GPU can read: device memory, or
 *               page-locked host memory (cudaHostAlloc / torch pin_memory -- the kernels then pull the packets over
 *               PCIe themselves and no separate host-to-device copy of the ring is needed).  16-byte aligned.
 *               BORROWED until `cuda_stream` has passed this call.  May be NULL if n_packets == 0.
 *   seq0        sequence number of the frame's first time sample; the frame holds samples [seq0, seq0 + T).
 *   frame_dev   OUT device uint8[T][F][N], 16-byte aligned: every position holds "good data or zeros";
 *               the voltage byte of every flagged sample is zeroed as well (reading P5), so the frame
 *               can go straight to xcorr_process().
 *   flags_dev   OUT device uint8[T][F][N/8], 16-byte aligned: the flag bit-field in the layout xcorr_norm_process()
 *               takes; zero where the packet is missing.  May be NULL.
 *   lost_dev    OUT device int32[F]: time samples of each channel lost with their packets in this frame (the
 *               paper's packet-loss counter, P6), ready for xcorr_norm_process_dev().  May be NULL.
 *   counts_dev  OUT device uint32[4], may be NULL: {packets kept, duplicates ignored, packets rejected, positions
 *               lost}.  A packet is rejected if its magic is wrong, its stream_id >= F / C, or its seq is outside
 *               [seq0, seq0 + T) or not a multiple of S away from seq0 (P3: it belongs to another frame or stream).
 *               Of several packets claiming one position the FIRST in arrival order is kept (P4).
 *
 * Two kernels: packet_claim_kernel (headers -> position ownership, lowest arrival index wins) and
 * assemble_kernel (one pass over the positions: copy / zero-fill, flag masking, footers, loss counters).
 * Errors: EINVAL (NULL / misaligned pointers, n_packets > 2^31 - 2), ECUDA.
 */
int xcorr_assemble(xcorr_assembler *a, const void *packets, size_t n_packets, uint64_t seq0, void *frame_dev,
                   uint8_t *flags_dev, int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream);

/*
 * xcorr_assemble_accounted -- xcorr_assemble() and xcorr_norm_process_dev() in ONE pass over the packets: the F-engine
 * flags of the footers ("the bit-field ... is read initially as 32-bit integers, and bit-field extraction is performed
 * only if ... non-zero") are counted into the handle's flag / intersection accumulator while they pass
 * through assemble_kernel's registers, and the packet-loss counters (:113, :115) go straight into the handle's.  The flag
 * field need not exist in memory at all: `flags_dev` and `lost_dev` are optional outputs here (NULL to skip).
 *
 *   h   a handle of the same N, F, T on the same device with xcorr_norm_enable() done; its accumulators are added to on
 *       `cuda_stream` (stream order with the handle's other calls as described in xcorr.h).
 * Everything else as in xcorr_assemble().  Errors: EINVAL (also: normalisation not enabled, shapes differ), ECUDA.
 */
int xcorr_assemble_accounted(xcorr_assembler *a, xcorr_handle *h, const void *packets, size_t n_packets, uint64_t seq0,
                             void *frame_dev, uint8_t *flags_dev, int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream);

/*
 * xcorr_assemble_static -- xcorr_assemble() for callers that must not allocate.  Same operation (PAPER.md:65-:81), same
 * kernels, same outputs byte for byte; what differs is where the scratch memory lives.
 *
 * Who needs it.  The paper's pipeline allocates everything at start-up and nothing afterwards ("the entire application
 * does not malloc or free any memory outside of startup and shutdown"), and a running acquisition has good
 * reason: cudaMalloc and cudaFree serialise against the whole device, so one call from any thread stalls the
 * correlation kernels of every stream in the middle of an integration.  A per-frame worker thread of such a pipeline
 * that was never handed an xcorr_assembler (a stream added, a frame length changed while the system runs) has no
 * permitted way to make one.  The other case is a process whose device memory is already spoken for by another
 * allocator (a PyTorch caching pool that has taken the card, a fixed partition handed out by a supervisor): a driver
 * allocation from inside this library can fail there or break the budget.  xcorr_assembler_create() allocates the position-ownership tables and the
 * counters with cudaMalloc; this call needs neither a handle nor an allocation.
 *
 * How.  The ownership tables and counters sit in one array that is part of libxcorr.so's device image (a file-scope
 * __device__ array of XCORR_ASSEMBLE_STATIC_SCRATCH_BYTES = 1 MiB + 256 B).  Every GPU on which the library's kernels
 * get loaded holds that array until the process exits, whether this call is ever used or not.  It bounds the frame:
 *
 *     (T / S) * (F / C)  <=  XCORR_ASSEMBLE_STATIC_MAX_POSITIONS  (131072 packet positions per frame;
 *                                                                   the paper's 256 MiB frame has 32768)
 *
 * A larger frame is refused with XCORR_ELIMIT before anything is enqueued; nothing is ever allocated to make it fit.
 *
 *   n_inputs, n_freq, t_per_frame, samples_per_packet, freq_per_packet
 *               the shapes xcorr_assembler_create() takes, with the same rules (N % 16 == 0, T % S == 0, F % C == 0,
 *               C * N a multiple of 128), checked on every call -- there is no handle to remember them.
 *   packets, n_packets, seq0, frame_dev, flags_dev, lost_dev, counts_dev, cuda_stream
 *               exactly as for xcorr_assemble(); all pointers belong to the CURRENT device.  The caller owns inputs and
 *               outputs; the library owns only the built-in scratch.
 *
 * Per call, on `cuda_stream`: two cudaMemsetAsync (the part of the ownership table this frame uses -> "no owner", the
 * counters -> 0), then packet_claim_kernel and assemble_kernel.  The call makes no cudaMalloc, cudaMallocHost,
 * cudaFree, stream / event creation or any other allocating call, first call included, and builds no host tables.
 *
 * First call on a device.  It looks up the device address of the built-in array (cudaGetSymbolAddress -- the name of a
 * __device__ array means nothing to host code until that is done, per device, with that device current), reads the SM
 * count and checks the architecture, and remembers all three for the process's lifetime.  This forces the library's
 * device code to be loaded onto that GPU if it was not yet.  Make this first call during start-up, and before any
 * stream capture is begun: a frame with n_packets = 0 is enough.
 *
 * Shared state -- read this.  There is ONE scratch array per device, shared by every caller in the process, and it
 * keeps whatever the last call left in it.  Each call clears what it needs at its own start, in stream order, so calls
 * one after another on one stream, or on streams the caller has ordered with events, are independent of each other and
 * of their shapes.  Two calls whose kernels may run at the same time on one GPU (different streams without such
 * ordering, different host threads each on its own stream) trample each other's ownership tables and counters: the
 * frames and counts that come out are garbage and nothing reports it.  Callers that need concurrent assembly on one GPU
 * create one xcorr_assembler per stream at start-up instead.  xcorr_assembler handles have their own tables and are
 * not affected by this call.
 *
 * Errors: EINVAL (shape rules, NULL / misaligned pointers, n_packets > 2^31 - 2), ELIMIT (more positions than the
 * built-in table holds), EARCH (current device is not sm_100), ECUDA (xcorr_assemble_static_last_cuda_error() has the
 * CUDA code).
 */
#define XCORR_ASSEMBLE_STATIC_MAX_POSITIONS 131072
#define XCORR_ASSEMBLE_STATIC_SCRATCH_BYTES (2 * 4 * XCORR_ASSEMBLE_STATIC_MAX_POSITIONS + 256)
int xcorr_assemble_static(int n_inputs, int n_freq, int t_per_frame, int samples_per_packet, int freq_per_packet,
                          const void *packets, size_t n_packets, uint64_t seq0, void *frame_dev, uint8_t *flags_dev,
                          int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream);

/* CUDA error code behind the calling thread's most recent XCORR_ECUDA from xcorr_assemble_static (0 if none). */
int xcorr_assemble_static_last_cuda_error(void);

/* Total number of this library's kernels launched through the assembler so far. */
uint64_t xcorr_assembler_kernel_launches(const xcorr_assembler *a);

/* Release everything (synchronises the device first).  NULL is a no-op. */
void xcorr_assembler_destroy(xcorr_assembler *a);

/*
 * xcorr_norm_process_dev -- xcorr_norm_process() (xcorr.h) with the packet-loss counters on the DEVICE, so that the
 * outputs of xcorr_assemble() feed the normalisation without a round trip through the host:
 *
 *   flags_dev          as in xcorr_norm_process (may be NULL)
 *   lost_samples_dev   device int32[F], added on `cuda_stream` to the handle's per-channel counters (may be NULL);
 *                      BORROWED until the stream has passed this call.
 * Errors: EINVAL (normalisation not enabled, misaligned), ECUDA.
 */
int xcorr_norm_process_dev(xcorr_handle *h, const uint8_t *flags_dev, const int32_t *lost_samples_dev, void *cuda_stream);

/* ---------------------------------------------------------------------------------------------------
 * Streamed packet path: what one server of the paper does per frame (Fig. 2, :47, :63) -- packets in a
 * page-locked host ring -> copy to the GPU -> assemble -> correlate -> (flag / loss accounting) -- on the two
 * streams of an xcorr_stream (xcorr.h, row a5), the copy of frame k+1's packets overlapping the kernels of frame k.
 * ------------------------------------------------------------------------------------------------- */

/*
 * xcorr_stream_attach_assembler -- startup-time call: gives the stream's `depth` ring slots a device buffer for
 * `max_packets` packets.  `a` (same N, F, T as the stream's handle) is BORROWED
 * until the stream is destroyed.  Once per stream.  Errors: EINVAL, ENOMEM.
 */
int xcorr_stream_attach_assembler(xcorr_stream *s, xcorr_assembler *a, size_t max_packets);

/*
 * xcorr_stream_submit_packets -- enqueue one frame given as its packets in arrival order (page-locked host memory,
 * n_packets <= max_packets, layout as for xcorr_assemble): H2D copy on the copy stream, then on the compute stream
 * xcorr_assemble -> xcorr_process; if the handle has normalisation enabled the assembly is xcorr_assemble_accounted, i.e.
 * the frame's flags and packet losses are accounted in the same pass.  `packets_host` is BORROWED until the copy has completed (as in
 * xcorr_stream_submit).  Returns without waiting unless all ring slots are in flight.
 * Errors: EINVAL, EOVERFLOW, ECUDA.
 */
int xcorr_stream_submit_packets(xcorr_stream *s, const void *packets_host, size_t n_packets, uint64_t seq0);

/* xcorr_read_normalized() ordered after all submitted frames on the compute stream; returns after the data has landed. */
int xcorr_stream_read_normalized(xcorr_stream *s, float *vis_out, int32_t *lost_matrix_out);

#ifdef __cplusplus
}
#endif
#endif /* XCORR_ASSEMBLE_H_ */
