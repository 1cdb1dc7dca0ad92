// xcorr_api.cu -- the C ABI declared in include/xcorr.h: handle management, work schedule, launches.
// All arithmetic of the hot path runs in the kernels of xengine_kernel.cuh / finalize_kernel.cuh.
#include "../../include/xcorr.h"
#include "../../include/xcorr_debug.h"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/xcorr_assemble.h"
#include "assemble_kernel.cuh"
#include "finalize_kernel.cuh"
#include "layout.hpp"
#include "normalise_kernel.cuh"
#include "schedule.hpp"
#include "xengine_kernel.cuh"

using namespace xc;

typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

constexpr unsigned long long kMaxTiles = 1ull << 18;

struct xcorr_handle {
    int n_inputs = 0, n_freq = 0, n_time = 0;
    int device = 0;
    int n_workers = 0;
    int n_sms = 0;
    int n_tiles = 0;                 // F * n_supertiles
    Segment head[kMaxHeadWorkers];   // first segment of every worker, copied into KernelParams at each launch
    bool offdiag = false;            // N > 256: kernel variant with the column block and -Im plane
    size_t frame_bytes = 0, output_bytes = 0, acc_bytes = 0;
    int32_t *acc = nullptr;          // device accumulator slots (layout.hpp), one per work segment
    int32_t *sums = nullptr;         // device column-sum slots (layout.hpp), one per work segment
    size_t sums_bytes = 0;
    unsigned long long offset_samples = 0;  // zero-padded samples the tensor path integrated since the last read (offset removal)
    int32_t *tile_slot_begin = nullptr;  // device, n_tiles + 1
    int n_slots = 0;
    bool clean = true;               // no frame since create / the last read: the next epilogue stores instead of adding
    bool frames_complete = false;    // xcorr_promise_complete_frames
    int32_t *staging = nullptr;      // device packed triangle for host reads
    Segment *segments = nullptr;     // device
    int32_t *worker_begin = nullptr; // device
    long long samples_since_read = 0;
    uint64_t launches = 0;
    int last_cuda_error = 0;
    PFN_encodeTiled encode = nullptr;
    // lost-sample normalisation (xcorr_norm_enable): flag-intersection accumulator, packet-loss counters
    bool norm = false;
    int32_t *flag_x = nullptr;       // device int32[F][P]: flag intersections (i < j)
    int32_t *flag_cnt = nullptr;     // device int32[2][F][N]: flag counters, double-buffered by integration (finalize_kernel.cuh)
    int32_t *lost_dev_acc = nullptr; // device int32[2][F]: packet-loss counters, double-buffered the same way
    int norm_half = 0;               // the half the current integration counts into
    bool lost_dev_dirty = false;
    int32_t *lost_pinned = nullptr;  // page-locked, device-mapped int32[2][F]: snapshots of lost_acc that lost_add_kernel
                                     // reads in place (no copy-engine operation in the stream); snapshot r uses half r % 2
    unsigned long long norm_reads = 0;
    long long *lost_acc = nullptr;   // host: lost samples per channel since the last read (xcorr_norm_process)
    bool lost_host_dirty = false;    // lost_acc holds counts of the current integration
    int32_t *staging_lost = nullptr; // device int32[F][P] for host reads of the normalisation matrix
    cudaEvent_t lost_used[2] = {nullptr, nullptr};   // recorded after the finalize launch that read the snapshot half
    bool flags_dirty = false;        // flag_x holds counts of the current integration
    // stream ordering of the handle's device state (accumulator slots, flag / loss accumulators): the stream of the last
    // call that enqueued work on them; a call on another stream first waits (on the device) for that work
    cudaStream_t last_stream = nullptr;
    bool has_last_stream = false;
    cudaEvent_t order_event = nullptr;
};

struct xcorr_stream {
    xcorr_handle *h = nullptr;
    int depth = 0;
    uint8_t *buf[8] = {};
    cudaEvent_t copied[8] = {}, consumed[8] = {};
    cudaStream_t copy_stream = nullptr, compute_stream = nullptr;
    unsigned long long submitted = 0;
    // packet path (xcorr_stream_attach_assembler): per ring slot a device copy of the packets, the flag field and the counters
    struct xcorr_assembler *assembler = nullptr;   // borrowed
    size_t max_packets = 0;
    uint8_t *pkt_buf[8] = {};
};

#define XC_CUDA(h, expr)                                  \
    do {                                                  \
        cudaError_t e_ = (expr);                          \
        if (e_ != cudaSuccess) {                          \
            if (h) (h)->last_cuda_error = (int)e_;        \
            return e_ == cudaErrorMemoryAllocation ? XCORR_ENOMEM : XCORR_ECUDA; \
        }                                                 \
    } while (0)

extern "C" const char *xcorr_strerror(int code)
{
    switch (code) {
        case XCORR_OK: return "ok";
        case XCORR_EINVAL: return "invalid argument";
        case XCORR_EARCH: return "current CUDA device is not compute capability 10.x (B200, sm_100a)";
        case XCORR_ENOMEM: return "out of memory";
        case XCORR_ECUDA: return "CUDA call failed (see xcorr_last_cuda_error)";
        case XCORR_EOVERFLOW: return "integration too long: an int32 visibility could overflow";
        case XCORR_ELIMIT: return "frame has more packet positions than the built-in scratch table holds (xcorr_assemble_static)";
        default: return "unknown xcorr error code";
    }
}

extern "C" int xcorr_last_cuda_error(const xcorr_handle *h) { return h ? h->last_cuda_error : 0; }
extern "C" size_t xcorr_frame_bytes(const xcorr_handle *h) { return h ? h->frame_bytes : 0; }
extern "C" size_t xcorr_output_bytes(const xcorr_handle *h) { return h ? h->output_bytes : 0; }
extern "C" uint64_t xcorr_kernel_launches(const xcorr_handle *h) { return h ? h->launches : 0; }

static int validate_shape(int n_inputs, int n_freq, int t_per_frame)
{
    if (n_inputs <= 0 || n_freq <= 0 || t_per_frame <= 0) return XCORR_EINVAL;
    if (n_inputs % 16 != 0) return XCORR_EINVAL;
    if (n_inputs > 65536 || n_freq > 65535) return XCORR_EINVAL;
    const unsigned long long bytes = (unsigned long long)n_inputs * (unsigned long long)n_freq * (unsigned long long)t_per_frame;
    if (bytes > (1ull << 40)) return XCORR_EINVAL;
    // work items (256 x 256 super-tiles): every one owns at least one 512 KiB accumulator slot, and the schedule tables
    // are built on the host -- refuse shapes whose tables alone would not fit a B200 (kMaxTiles slots = 128 GiB)
    const unsigned long long nb = ((unsigned long long)n_inputs + kSuper - 1) / kSuper;
    const unsigned long long tiles = (unsigned long long)n_freq * (nb * (nb + 1) / 2);
    if (tiles > kMaxTiles) return XCORR_EINVAL;
    return XCORR_OK;
}

// make_schedule builds std::vectors: never let an exception cross the C ABI
static int make_schedule_noexcept(int n_inputs, int n_freq, int t_per_frame, int n_workers, Schedule *out)
{
    try {
        *out = make_schedule(n_inputs, n_freq, t_per_frame, n_workers);
    } catch (...) {
        return XCORR_ENOMEM;
    }
    return XCORR_OK;
}

// The handle's device pointers belong to the device that was current at xcorr_create()
static int check_device(int device)
{
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) return XCORR_ECUDA;
    return cur == device ? XCORR_OK : XCORR_EINVAL;
}

// Order this call's work after the handle's previous work.  Same stream as last time: stream order does it (and nothing
// is put between two kernels, so programmatic dependent launch keeps working).  Another stream: record an event behind
// everything enqueued so far on the previous stream and make the new stream wait for it on the device.
static int order_after_previous(xcorr_handle *h, cudaStream_t s)
{
    if (h->has_last_stream && h->last_stream != s) {
        cudaError_t e = cudaEventRecord(h->order_event, h->last_stream);
        if (e != cudaSuccess) { cudaGetLastError(); h->last_cuda_error = (int)e; return XCORR_EINVAL; }   // e.g. that stream was destroyed
        XC_CUDA(h, cudaStreamWaitEvent(s, h->order_event, 0));
    }
    h->last_stream = s;
    h->has_last_stream = true;
    return XCORR_OK;
}

extern "C" void xcorr_destroy(xcorr_handle *h)
{
    if (!h) return;
    cudaSetDevice(h->device);
    cudaDeviceSynchronize();
    cudaFree(h->acc);
    cudaFree(h->sums);
    cudaFree(h->staging);
    cudaFree(h->segments);
    cudaFree(h->worker_begin);
    cudaFree(h->tile_slot_begin);
    cudaFree(h->flag_x);
    cudaFree(h->lost_dev_acc);
    cudaFree(h->flag_cnt);
    cudaFree(h->staging_lost);
    if (h->lost_pinned) cudaFreeHost(h->lost_pinned);
    if (h->order_event) cudaEventDestroy(h->order_event);
    for (int k = 0; k < 2; ++k)
        if (h->lost_used[k]) cudaEventDestroy(h->lost_used[k]);
    delete[] h->lost_acc;
    delete h;
}

extern "C" int xcorr_create(int n_inputs, int n_freq, int t_per_frame, xcorr_handle **out)
{
    if (!out) return XCORR_EINVAL;
    *out = nullptr;
    int rc = validate_shape(n_inputs, n_freq, t_per_frame);
    if (rc != XCORR_OK) return rc;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return XCORR_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return XCORR_ECUDA;
    if (prop.major != 10) return XCORR_EARCH;

    xcorr_handle *h = new (std::nothrow) xcorr_handle;
    if (!h) return XCORR_ENOMEM;
    h->n_inputs = n_inputs;
    h->n_freq = n_freq;
    h->n_time = t_per_frame;
    h->device = dev;
    h->frame_bytes = (size_t)n_inputs * n_freq * t_per_frame;
    h->output_bytes = (size_t)n_freq * ((size_t)n_inputs * (n_inputs + 1) / 2) * 8;
    const int nb = n_super(n_inputs);
    h->n_tiles = n_freq * n_supertiles(nb);
    h->offdiag = nb > 1;
    h->n_sms = prop.multiProcessorCount;
    h->n_workers = prop.multiProcessorCount / 2;
    if (h->n_workers < 1) { delete h; return XCORR_EARCH; }

    auto fail = [&](int code) { xcorr_destroy(h); return code; };

    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return fail(XCORR_ECUDA);
    h->encode = (PFN_encodeTiled)fn;

    Schedule sched;
    if ((rc = make_schedule_noexcept(n_inputs, n_freq, t_per_frame, h->n_workers, &sched)) != XCORR_OK) return fail(rc);
    if (cudaEventCreateWithFlags(&h->order_event, cudaEventDisableTiming) != cudaSuccess) return fail(XCORR_ECUDA);
    for (int w = 0; w < kMaxHeadWorkers; ++w) {   // KernelParams::head: the first segment of every worker
        h->head[w] = Segment{};
        if (w < h->n_workers && sched.worker_begin[w] < sched.worker_begin[w + 1]) h->head[w] = sched.segments[sched.worker_begin[w]];
    }
    h->n_slots = (int)sched.segments.size();
    h->acc_bytes = (size_t)h->n_slots * kAccElemsPerSlot * sizeof(int32_t);
    cudaError_t e;
    if ((e = cudaMalloc(&h->acc, h->acc_bytes)) != cudaSuccess) { h->last_cuda_error = e; return fail(XCORR_ENOMEM); }
    h->sums_bytes = (size_t)h->n_slots * kSumElemsPerSlot * sizeof(int32_t);
    if ((e = cudaMalloc(&h->sums, h->sums_bytes)) != cudaSuccess) { h->last_cuda_error = e; return fail(XCORR_ENOMEM); }
    if (cudaMemset(h->sums, 0, h->sums_bytes) != cudaSuccess) return fail(XCORR_ECUDA);
    if ((e = cudaMalloc(&h->staging, h->output_bytes)) != cudaSuccess) { h->last_cuda_error = e; return fail(XCORR_ENOMEM); }
    if ((e = cudaMalloc(&h->segments, sizeof(Segment) * (sched.segments.size() + 1))) != cudaSuccess) return fail(XCORR_ENOMEM);
    if ((e = cudaMalloc(&h->worker_begin, sizeof(int32_t) * sched.worker_begin.size())) != cudaSuccess) return fail(XCORR_ENOMEM);
    if ((e = cudaMalloc(&h->tile_slot_begin, sizeof(int32_t) * sched.tile_slot_begin.size())) != cudaSuccess) return fail(XCORR_ENOMEM);
    if (cudaMemset(h->acc, 0, h->acc_bytes) != cudaSuccess) return fail(XCORR_ECUDA);
    if (cudaMemcpy(h->tile_slot_begin, sched.tile_slot_begin.data(), sizeof(int32_t) * sched.tile_slot_begin.size(),
                   cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(XCORR_ECUDA);
    if (!sched.segments.empty() &&
        cudaMemcpy(h->segments, sched.segments.data(), sizeof(Segment) * sched.segments.size(), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(XCORR_ECUDA);
    if (cudaMemcpy(h->worker_begin, sched.worker_begin.data(), sizeof(int32_t) * sched.worker_begin.size(), cudaMemcpyHostToDevice) !=
        cudaSuccess)
        return fail(XCORR_ECUDA);

    if (h->offdiag)
        e = cudaFuncSetAttribute(xengine_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, KernelCfg<true>::kSmemBytes);
    else
        e = cudaFuncSetAttribute(xengine_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, KernelCfg<false>::kSmemBytes);
    if (e != cudaSuccess) { h->last_cuda_error = e; return fail(XCORR_ECUDA); }
    if (cudaDeviceSynchronize() != cudaSuccess) return fail(XCORR_ECUDA);
    *out = h;
    return XCORR_OK;
}

static int encode_frame_map(xcorr_handle *h, const void *frame_dev, CUtensorMap *map)
{
    // a1: global uint8[T][F][N] seen as a 3-D tensor (n, f, t); one box = 128 inputs x 1 channel x kStageT samples,
    // written to smem as kStageT rows of 128 bytes with the 128-byte swizzle the MMA descriptors expect.
    const cuuint64_t dims[3] = {(cuuint64_t)h->n_inputs, (cuuint64_t)h->n_freq, (cuuint64_t)h->n_time};
    const cuuint64_t strides[2] = {(cuuint64_t)h->n_inputs, (cuuint64_t)h->n_inputs * (cuuint64_t)h->n_freq};
    const cuuint32_t box[3] = {(cuuint32_t)kBlock, 1u, (cuuint32_t)kStageT};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = h->encode(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(frame_dev), dims, strides, box, estr,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->last_cuda_error = (int)r;
        return XCORR_ECUDA;
    }
    return XCORR_OK;
}

static int check_process_args(xcorr_handle *h, const void *frame)
{
    if (!h || !frame) return XCORR_EINVAL;
    if (((uintptr_t)frame & 15u) != 0) return XCORR_EINVAL;
    // |sum| <= 128 * samples must stay <= 2^31 - 1
    if (h->samples_since_read + (long long)h->n_time > 16777215ll) return XCORR_EOVERFLOW;
    return XCORR_OK;
}

extern "C" int xcorr_process(xcorr_handle *h, const void *packed_frame_dev, void *cuda_stream)
{
    int rc = check_process_args(h, packed_frame_dev);
    if (rc != XCORR_OK) return rc;
    if ((rc = check_device(h->device)) != XCORR_OK) return rc;
    alignas(64) CUtensorMap map;
    rc = encode_frame_map(h, packed_frame_dev, &map);
    if (rc != XCORR_OK) return rc;
    if ((rc = order_after_previous(h, (cudaStream_t)cuda_stream)) != XCORR_OK) return rc;
    KernelParams p;
    for (int w = 0; w < kMaxHeadWorkers; ++w) p.head[w] = h->head[w];
    p.segments = h->segments;
    p.worker_begin = h->worker_begin;
    p.acc = h->acc;
    p.sums = h->sums;
    p.first_frame = h->clean ? 1 : 0;
    p.n_inputs = h->n_inputs;
    p.n_freq = h->n_freq;
    p.n_time = h->n_time;
    p.wait_frame = h->frames_complete ? 0 : 1;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // programmatic dependent launch: this kernel's prologue (barrier init, TMEM allocation, cluster sync) may overlap the
    // tail of the previous kernel of the stream; the kernel itself waits (griddepcontrol.wait) before touching memory
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * h->n_workers);
    cfg.stream = s;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (h->offdiag) {
        cfg.blockDim = dim3(KernelCfg<true>::kThreads);
        cfg.dynamicSmemBytes = KernelCfg<true>::kSmemBytes;
        XC_CUDA(h, cudaLaunchKernelEx(&cfg, xengine_kernel<true>, map, p));
    } else {
        cfg.blockDim = dim3(KernelCfg<false>::kThreads);
        cfg.dynamicSmemBytes = KernelCfg<false>::kSmemBytes;
        XC_CUDA(h, cudaLaunchKernelEx(&cfg, xengine_kernel<false>, map, p));
    }
    XC_CUDA(h, cudaGetLastError());
    h->launches += 1;
    h->samples_since_read += h->n_time;
    h->offset_samples += (unsigned long long)((h->n_time + kStageT - 1) / kStageT) * kStageT;   // TMA zero fill = samples of value 0
    h->clean = false;
    return XCORR_OK;
}

static bool is_device_pointer(const void *ptr)
{
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, ptr) == cudaSuccess) return attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged;
    cudaGetLastError();
    return false;
}

// xcorr_read / xcorr_read_normalized: one launch of finalize_kernel; ends the integration
static int read_common(xcorr_handle *h, void *vis_out, bool normalise, int32_t *lost_matrix_out, void *cuda_stream, bool wait = true)
{
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int rc0 = check_device(h->device);
    if (rc0 != XCORR_OK) return rc0;
    const bool on_device = is_device_pointer(vis_out);
    if (on_device && ((uintptr_t)vis_out & 15u) != 0) return XCORR_EINVAL;
    if ((rc0 = order_after_previous(h, s)) != XCORR_OK) return rc0;
    void *dst = on_device ? vis_out : (void *)h->staging;
    const bool lost_on_device = lost_matrix_out && is_device_pointer(lost_matrix_out);
    int32_t *lost_dst = !lost_matrix_out ? nullptr : (lost_on_device ? lost_matrix_out : h->staging_lost);
    const int nt = (h->n_inputs + 31) / 32;
    const size_t lost_matrix_bytes = h->output_bytes / 2;
    if (h->clean) {   // nothing integrated: the result is all zeros
        XC_CUDA(h, cudaMemsetAsync(h->acc, 0, h->acc_bytes, s));
        XC_CUDA(h, cudaMemsetAsync(h->sums, 0, h->sums_bytes, s));
    }
    NormParams np = {};
    if (normalise) {
        const size_t cnt_half = (size_t)h->n_freq * h->n_inputs;
        int32_t *lost_cur = h->lost_dev_acc + (size_t)h->norm_half * h->n_freq;
        if (h->lost_host_dirty) {
            // packet-loss counters tallied on the host (xcorr_norm_process): a page-locked snapshot the device adds in place; a
            // snapshot half is reused two such reads later, after the event recorded behind its reader
            const int snap_half = (int)(h->norm_reads++ & 1u);
            XC_CUDA(h, cudaEventSynchronize(h->lost_used[snap_half]));
            int32_t *snap = h->lost_pinned + (size_t)snap_half * h->n_freq;
            for (int f = 0; f < h->n_freq; ++f) snap[f] = (int32_t)h->lost_acc[f];
            lost_add_kernel<<<(h->n_freq + 255) / 256, 256, 0, s>>>(snap, lost_cur, h->n_freq);
            XC_CUDA(h, cudaGetLastError());
            h->launches += 1;
            XC_CUDA(h, cudaEventRecord(h->lost_used[snap_half], s));
        }
        np.x = h->flag_x;
        np.cnt = h->flag_cnt + (size_t)h->norm_half * cnt_half;
        np.cnt_clear = h->flag_cnt + (size_t)(h->norm_half ^ 1) * cnt_half;
        np.lost = lost_cur;
        np.lost_clear = h->lost_dev_acc + (size_t)(h->norm_half ^ 1) * h->n_freq;
        np.lost_out = lost_dst;
        np.n_samples = (uint32_t)h->samples_since_read;
    }
    {
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(nt, nt, h->n_freq);
        cfg.blockDim = dim3(256);
        cfg.stream = s;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (normalise)
            XC_CUDA(h, cudaLaunchKernelEx(&cfg, finalize_kernel<true>, (const int32_t *)h->acc, (const int32_t *)h->sums,
                                          (const int32_t *)h->tile_slot_begin, dst, h->n_inputs, (uint32_t)h->offset_samples, np));
        else
            XC_CUDA(h, cudaLaunchKernelEx(&cfg, finalize_kernel<false>, (const int32_t *)h->acc, (const int32_t *)h->sums,
                                          (const int32_t *)h->tile_slot_begin, dst, h->n_inputs, (uint32_t)h->offset_samples, np));
    }
    XC_CUDA(h, cudaGetLastError());
    h->launches += 1;
    // ends the integration: no clearing pass over the visibilities -- the next frame's epilogue overwrites its slots
    h->samples_since_read = 0;
    h->offset_samples = 0;
    h->clean = true;
    if (h->norm) {   // the flag / loss state belongs to the integration that just ended
        if (normalise) {
            // finalize_kernel<true> has cleared the intersections it read and the OTHER half of the counters: that half is the
            // next integration's
            h->norm_half ^= 1;
        } else {
            const size_t cnt_half = (size_t)h->n_freq * h->n_inputs;
            if (h->flags_dirty) {
                XC_CUDA(h, cudaMemsetAsync(h->flag_x, 0, lost_matrix_bytes, s));
                XC_CUDA(h, cudaMemsetAsync(h->flag_cnt + (size_t)h->norm_half * cnt_half, 0, sizeof(int32_t) * cnt_half, s));
            }
            if (h->lost_dev_dirty)
                XC_CUDA(h, cudaMemsetAsync(h->lost_dev_acc + (size_t)h->norm_half * h->n_freq, 0, sizeof(int32_t) * h->n_freq, s));
        }
        h->flags_dirty = false;
        h->lost_dev_dirty = false;
        if (h->lost_host_dirty)
            for (int f = 0; f < h->n_freq; ++f) h->lost_acc[f] = 0;
        h->lost_host_dirty = false;
    }
    if (!on_device) XC_CUDA(h, cudaMemcpyAsync(vis_out, h->staging, h->output_bytes, cudaMemcpyDeviceToHost, s));
    if (lost_matrix_out && !lost_on_device)
        XC_CUDA(h, cudaMemcpyAsync(lost_matrix_out, h->staging_lost, lost_matrix_bytes, cudaMemcpyDeviceToHost, s));
    if (wait && (!on_device || (lost_matrix_out && !lost_on_device))) XC_CUDA(h, cudaStreamSynchronize(s));
    return XCORR_OK;
}

extern "C" int xcorr_promise_complete_frames(xcorr_handle *h, int enabled)
{
    if (!h) return XCORR_EINVAL;
    h->frames_complete = enabled != 0;
    return XCORR_OK;
}

extern "C" int xcorr_read(xcorr_handle *h, int32_t *upper_triangle_out, void *cuda_stream)
{
    if (!h || !upper_triangle_out) return XCORR_EINVAL;
    return read_common(h, upper_triangle_out, false, nullptr, cuda_stream);
}

// ---------------------------------------------------------------------------------------------------
// lost-sample normalisation (NEXT-1)
// ---------------------------------------------------------------------------------------------------
extern "C" int xcorr_norm_enable(xcorr_handle *h)
{
    if (!h) return XCORR_EINVAL;
    if (h->norm) return XCORR_OK;
    if (!h->clean) return XCORR_EINVAL;   // startup-time call: not in the middle of an integration
    int rc = check_device(h->device);
    if (rc != XCORR_OK) return rc;
    const size_t lost_matrix_bytes = h->output_bytes / 2;
    // everything or nothing: a failure frees what this call allocated, so a retry starts from scratch
    auto undo = [&](int code, cudaError_t e) {
        if (e != cudaSuccess) { h->last_cuda_error = (int)e; cudaGetLastError(); }
        cudaFree(h->flag_x); h->flag_x = nullptr;
        cudaFree(h->staging_lost); h->staging_lost = nullptr;
        cudaFree(h->flag_cnt); h->flag_cnt = nullptr;
        cudaFree(h->lost_dev_acc); h->lost_dev_acc = nullptr;
        if (h->lost_pinned) cudaFreeHost(h->lost_pinned);
        h->lost_pinned = nullptr;
        delete[] h->lost_acc; h->lost_acc = nullptr;
        for (int k = 0; k < 2; ++k) {
            if (h->lost_used[k]) cudaEventDestroy(h->lost_used[k]);
            h->lost_used[k] = nullptr;
        }
        return code;
    };
    cudaError_t e;
    if ((e = cudaMalloc(&h->flag_x, lost_matrix_bytes)) != cudaSuccess) return undo(XCORR_ENOMEM, e);
    if ((e = cudaMalloc(&h->staging_lost, lost_matrix_bytes)) != cudaSuccess) return undo(XCORR_ENOMEM, e);
    const size_t cnt_bytes = sizeof(int32_t) * 2 * (size_t)h->n_freq * h->n_inputs;
    if ((e = cudaMalloc(&h->flag_cnt, cnt_bytes)) != cudaSuccess) return undo(XCORR_ENOMEM, e);
    if ((e = cudaMalloc(&h->lost_dev_acc, sizeof(int32_t) * 2 * h->n_freq)) != cudaSuccess) return undo(XCORR_ENOMEM, e);
    if ((e = cudaMallocHost(&h->lost_pinned, sizeof(int32_t) * 2 * h->n_freq)) != cudaSuccess) return undo(XCORR_ENOMEM, e);
    h->lost_acc = new (std::nothrow) long long[h->n_freq]();
    if (!h->lost_acc) return undo(XCORR_ENOMEM, cudaSuccess);
    for (int k = 0; k < 2; ++k)
        if ((e = cudaEventCreateWithFlags(&h->lost_used[k], cudaEventDisableTiming)) != cudaSuccess) return undo(XCORR_ECUDA, e);
    if ((e = cudaMemset(h->flag_x, 0, lost_matrix_bytes)) != cudaSuccess) return undo(XCORR_ECUDA, e);
    if ((e = cudaMemset(h->flag_cnt, 0, cnt_bytes)) != cudaSuccess) return undo(XCORR_ECUDA, e);
    if ((e = cudaMemset(h->lost_dev_acc, 0, sizeof(int32_t) * 2 * h->n_freq)) != cudaSuccess) return undo(XCORR_ECUDA, e);
    h->norm_half = 0;
    h->norm = true;
    return XCORR_OK;
}

static int launch_flag_count(xcorr_handle *h, const uint8_t *flags_dev, void *cuda_stream);

extern "C" int xcorr_norm_process_dev(xcorr_handle *h, const uint8_t *flags_dev, const int32_t *lost_samples_dev, void *cuda_stream)
{
    if (!h || !h->norm) return XCORR_EINVAL;
    if (flags_dev && ((uintptr_t)flags_dev & 15u) != 0) return XCORR_EINVAL;
    int rc = check_device(h->device);
    if (rc != XCORR_OK) return rc;
    if ((flags_dev || lost_samples_dev) && (rc = order_after_previous(h, (cudaStream_t)cuda_stream)) != XCORR_OK) return rc;
    if (lost_samples_dev) {
        lost_add_kernel<<<(h->n_freq + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(lost_samples_dev, h->lost_dev_acc + (size_t)h->norm_half * h->n_freq,
                                                                                        h->n_freq);
        XC_CUDA(h, cudaGetLastError());
        h->launches += 1;
        h->lost_dev_dirty = true;
    }
    return launch_flag_count(h, flags_dev, cuda_stream);
}

extern "C" int xcorr_norm_process(xcorr_handle *h, const uint8_t *flags_dev, const int32_t *lost_samples_host, void *cuda_stream)
{
    if (!h || !h->norm) return XCORR_EINVAL;
    if (flags_dev && ((uintptr_t)flags_dev & 15u) != 0) return XCORR_EINVAL;
    if (lost_samples_host)
        for (int f = 0; f < h->n_freq; ++f)
            if (lost_samples_host[f] < 0 || lost_samples_host[f] > h->n_time) return XCORR_EINVAL;
    if (flags_dev) {
        int rc = check_device(h->device);
        if (rc != XCORR_OK) return rc;
        if ((rc = order_after_previous(h, (cudaStream_t)cuda_stream)) != XCORR_OK) return rc;
    }
    // the flag launch goes first: if it fails, the host-side loss counters have not moved and the caller may retry the
    // whole call without counting this frame's lost samples twice
    const int rc = launch_flag_count(h, flags_dev, cuda_stream);
    if (rc != XCORR_OK) return rc;
    if (lost_samples_host) {
        for (int f = 0; f < h->n_freq; ++f) h->lost_acc[f] += lost_samples_host[f];
        h->lost_host_dirty = true;
    }
    return XCORR_OK;
}

static int launch_flag_count(xcorr_handle *h, const uint8_t *flags_dev, void *cuda_stream)
{
    if (flags_dev) {
        const unsigned long long n_bytes = (unsigned long long)h->frame_bytes / 8;
        const unsigned long long n_pieces = (n_bytes + 16ull * 32 * kFlagUnroll - 1) / (16ull * 32 * kFlagUnroll);   // 2 KiB per warp and iteration
        int blocks = h->n_sms * 8;     // warp-stride, 8 resident CTAs of 256 threads (8 warps) per SM
        if ((unsigned long long)blocks * 8ull > n_pieces) blocks = (int)((n_pieces + 7) / 8);
        flag_count_kernel<<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>(flags_dev, n_bytes, h->n_inputs, h->n_freq, h->flag_x,
                                                                         h->flag_cnt + (size_t)h->norm_half * h->n_freq * h->n_inputs);
        XC_CUDA(h, cudaGetLastError());
        h->launches += 1;
        h->flags_dirty = true;
    }
    return XCORR_OK;
}

extern "C" int xcorr_read_normalized(xcorr_handle *h, float *vis_out, int32_t *lost_matrix_out, void *cuda_stream)
{
    if (!h || !vis_out || !h->norm) return XCORR_EINVAL;
    if (lost_matrix_out && is_device_pointer(lost_matrix_out) && ((uintptr_t)lost_matrix_out & 15u) != 0) return XCORR_EINVAL;
    return read_common(h, vis_out, true, lost_matrix_out, cuda_stream);
}

// ---------------------------------------------------------------------------------------------------
// streamed frame path (a5)
// ---------------------------------------------------------------------------------------------------
extern "C" void xcorr_stream_destroy(xcorr_stream *s)
{
    if (!s) return;
    if (s->h) cudaSetDevice(s->h->device);
    cudaDeviceSynchronize();
    // everything the handle enqueued has finished, and the compute stream is about to go: nothing left to order after
    if (s->h && s->h->has_last_stream && s->h->last_stream == s->compute_stream) s->h->has_last_stream = false;
    for (int k = 0; k < s->depth; ++k) {
        if (s->buf[k]) cudaFree(s->buf[k]);
        if (s->pkt_buf[k]) cudaFree(s->pkt_buf[k]);
        if (s->copied[k]) cudaEventDestroy(s->copied[k]);
        if (s->consumed[k]) cudaEventDestroy(s->consumed[k]);
    }
    if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
    if (s->compute_stream) cudaStreamDestroy(s->compute_stream);
    delete s;
}

extern "C" int xcorr_stream_create(xcorr_handle *h, int depth, xcorr_stream **out)
{
    if (!h || !out || depth < 2 || depth > 8) return XCORR_EINVAL;
    *out = nullptr;
    xcorr_stream *s = new (std::nothrow) xcorr_stream;
    if (!s) return XCORR_ENOMEM;
    s->h = h;
    s->depth = depth;
    auto fail = [&](int code) { xcorr_stream_destroy(s); return code; };
    if (cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(XCORR_ECUDA);
    if (cudaStreamCreateWithFlags(&s->compute_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(XCORR_ECUDA);
    for (int k = 0; k < depth; ++k) {
        if (cudaMalloc(&s->buf[k], h->frame_bytes) != cudaSuccess) return fail(XCORR_ENOMEM);
        if (cudaEventCreateWithFlags(&s->copied[k], cudaEventDisableTiming) != cudaSuccess) return fail(XCORR_ECUDA);
        if (cudaEventCreateWithFlags(&s->consumed[k], cudaEventDisableTiming) != cudaSuccess) return fail(XCORR_ECUDA);
    }
    *out = s;
    return XCORR_OK;
}

extern "C" int xcorr_stream_submit(xcorr_stream *s, const void *frame_host)
{
    if (!s || !frame_host) return XCORR_EINVAL;
    xcorr_handle *h = s->h;
    if (h->samples_since_read + (long long)h->n_time > 16777215ll) return XCORR_EOVERFLOW;
    const int k = (int)(s->submitted % (unsigned long long)s->depth);
    if (s->submitted >= (unsigned long long)s->depth) {
        // ring-buffer back-pressure: the correlation that last read this device buffer must have finished
        XC_CUDA(h, cudaEventSynchronize(s->consumed[k]));
    }
    XC_CUDA(h, cudaMemcpyAsync(s->buf[k], frame_host, h->frame_bytes, cudaMemcpyHostToDevice, s->copy_stream));
    XC_CUDA(h, cudaEventRecord(s->copied[k], s->copy_stream));
    XC_CUDA(h, cudaStreamWaitEvent(s->compute_stream, s->copied[k], 0));
    const int rc = xcorr_process(h, s->buf[k], (void *)s->compute_stream);
    if (rc != XCORR_OK) return rc;
    XC_CUDA(h, cudaEventRecord(s->consumed[k], s->compute_stream));
    s->submitted += 1;
    return XCORR_OK;
}

extern "C" int xcorr_stream_sync(xcorr_stream *s)
{
    if (!s) return XCORR_EINVAL;
    XC_CUDA(s->h, cudaStreamSynchronize(s->copy_stream));
    XC_CUDA(s->h, cudaStreamSynchronize(s->compute_stream));
    return XCORR_OK;
}

extern "C" int xcorr_stream_read(xcorr_stream *s, int32_t *upper_triangle_out)
{
    if (!s || !upper_triangle_out) return XCORR_EINVAL;
    const int rc = xcorr_read(s->h, upper_triangle_out, (void *)s->compute_stream);
    if (rc != XCORR_OK) return rc;
    XC_CUDA(s->h, cudaStreamSynchronize(s->compute_stream));
    return XCORR_OK;
}

extern "C" int xcorr_stream_read_async(xcorr_stream *s, int32_t *upper_triangle_out)
{
    if (!s || !upper_triangle_out) return XCORR_EINVAL;
    return read_common(s->h, upper_triangle_out, false, nullptr, (void *)s->compute_stream, /*wait=*/false);
}

// ---------------------------------------------------------------------------------------------------
// debug / test support (include/xcorr_debug.h) -- never on the xcorr_process path
// ---------------------------------------------------------------------------------------------------
extern "C" int xcorr_debug_schedule(int n_inputs, int n_freq, int t_per_frame, int n_workers, int32_t *segments_out, int max_segments,
                                    int32_t *worker_begin_out)
{
    if (validate_shape(n_inputs, n_freq, t_per_frame) != XCORR_OK || n_workers <= 0) return XCORR_EINVAL;
    Schedule sched;
    if (make_schedule_noexcept(n_inputs, n_freq, t_per_frame, n_workers, &sched) != XCORR_OK) return XCORR_ENOMEM;
    const int n = (int)sched.segments.size();
    if (segments_out && worker_begin_out) {
        if (n > max_segments) return XCORR_EINVAL;
        for (int k = 0; k < n; ++k) {
            const Segment &g = sched.segments[k];
            int32_t *o = segments_out + 7 * k;
            o[0] = g.f; o[1] = g.I; o[2] = g.J; o[3] = g.stage_begin; o[4] = g.stage_end; o[5] = g.tile; o[6] = g.slot;
        }
        for (int w = 0; w <= n_workers; ++w) worker_begin_out[w] = sched.worker_begin[w];
    }
    return n;
}

extern "C" int xcorr_debug_stage_samples(void) { return kStageT; }

// ---------------------------------------------------------------------------------------------------
// packet -> frame assembly (NEXT-2; include/xcorr_assemble.h)
// ---------------------------------------------------------------------------------------------------
struct xcorr_assembler {
    AssembleShape sh = {};
    int device = 0, n_sms = 0;
    unsigned n_positions = 0;
    uint32_t *owner = nullptr;     // device uint32[2][n_positions]: arrival index of the packet that owns the position; the
                                   // two tables alternate from call to call (assemble_kernel.cuh)
    unsigned long long calls = 0;
    uint32_t *counts = nullptr;    // device uint32[8], see assemble_kernel.cuh
    int ctas_per_sm[2] = {8, 8};   // resident CTAs of assemble_kernel<false> / <true> per SM: the grid-stride grid is exactly one wave
    uint64_t launches = 0;
    int last_cuda_error = 0;
};

extern "C" void xcorr_assembler_destroy(xcorr_assembler *a)
{
    if (!a) return;
    cudaSetDevice(a->device);
    cudaDeviceSynchronize();
    cudaFree(a->owner);
    cudaFree(a->counts);
    delete a;
}

extern "C" size_t xcorr_assembler_packet_bytes(const xcorr_assembler *a) { return a ? (size_t)a->sh.packet_bytes : 0; }
extern "C" uint64_t xcorr_assembler_kernel_launches(const xcorr_assembler *a) { return a ? a->launches : 0; }

extern "C" int xcorr_assembler_create(int n_inputs, int n_freq, int t_per_frame, int samples_per_packet, int freq_per_packet,
                                      xcorr_assembler **out)
{
    if (!out) return XCORR_EINVAL;
    *out = nullptr;
    int rc = validate_shape(n_inputs, n_freq, t_per_frame);
    if (rc != XCORR_OK) return rc;
    const int S = samples_per_packet, C = freq_per_packet;
    if (S <= 0 || C <= 0 || t_per_frame % S != 0 || n_freq % C != 0) return XCORR_EINVAL;
    if (((long long)C * n_inputs) % 128 != 0) return XCORR_EINVAL;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return XCORR_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return XCORR_ECUDA;
    if (prop.major != 10) return XCORR_EARCH;
    xcorr_assembler *a = new (std::nothrow) xcorr_assembler;
    if (!a) return XCORR_ENOMEM;
    a->device = dev;
    a->n_sms = prop.multiProcessorCount;
    a->sh.n_inputs = n_inputs; a->sh.n_freq = n_freq; a->sh.n_time = t_per_frame;
    a->sh.s_per_packet = S; a->sh.c_per_packet = C;
    a->sh.n_streams = n_freq / C; a->sh.n_blocks = t_per_frame / S;
    const unsigned long long pay = (unsigned long long)S * C * n_inputs;
    a->sh.packet_bytes = kPacketHeaderBytes + pay + pay / 8;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a->ctas_per_sm[0], assemble_kernel<false>, 256, 0) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a->ctas_per_sm[1], assemble_kernel<true>, 256, 0) != cudaSuccess ||
        a->ctas_per_sm[0] < 1 || a->ctas_per_sm[1] < 1) {
        cudaGetLastError();
        delete a;
        return XCORR_ECUDA;
    }
    const unsigned long long n_pos = (unsigned long long)a->sh.n_streams * (unsigned long long)a->sh.n_blocks;
    if (n_pos == 0 || n_pos > 0x7FFFFFFFull) { delete a; return XCORR_EINVAL; }
    a->n_positions = (unsigned)n_pos;
    cudaError_t e;
    if ((e = cudaMalloc(&a->owner, sizeof(uint32_t) * 2 * (size_t)a->n_positions)) != cudaSuccess ||
        (e = cudaMalloc(&a->counts, sizeof(uint32_t) * 8)) != cudaSuccess) {
        cudaGetLastError();
        xcorr_assembler_destroy(a);
        return e == cudaErrorMemoryAllocation ? XCORR_ENOMEM : XCORR_ECUDA;
    }
    if ((e = cudaMemset(a->owner, 0xFF, sizeof(uint32_t) * 2 * (size_t)a->n_positions)) != cudaSuccess ||
        (e = cudaMemset(a->counts, 0, sizeof(uint32_t) * 8)) != cudaSuccess) {
        xcorr_assembler_destroy(a);
        return XCORR_ECUDA;
    }
    *out = a;
    return XCORR_OK;
}

static int assemble_common(xcorr_assembler *a, xcorr_handle *h, const void *packets, size_t n_packets, uint64_t seq0, void *frame_dev,
                           uint8_t *flags_dev, int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream)
{
    if (!a || !frame_dev || (!packets && n_packets) || n_packets > 0x7FFFFFFEull) return XCORR_EINVAL;
    if (((uintptr_t)packets & 15u) || ((uintptr_t)frame_dev & 15u) || ((uintptr_t)flags_dev & 15u) || ((uintptr_t)lost_dev & 3u) ||
        ((uintptr_t)counts_dev & 3u))
        return XCORR_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    {
        const int rc = check_device(a->device);
        if (rc != XCORR_OK) return rc;
    }
    if (h) {   // accounted form: the handle's flag / loss accumulators are written by assemble_kernel on this stream
        if (!h->norm || h->device != a->device || h->n_inputs != a->sh.n_inputs || h->n_freq != a->sh.n_freq || h->n_time != a->sh.n_time)
            return XCORR_EINVAL;
        const int rc = order_after_previous(h, s);
        if (rc != XCORR_OK) return rc;
    }
    // no memsets: the ownership tables and counters are left clean by the previous call's assemble_kernel (see create)
    uint32_t *owner = a->owner + (size_t)(a->calls & 1u) * a->n_positions;
    uint32_t *owner_next = a->owner + (size_t)((a->calls + 1) & 1u) * a->n_positions;
    {
        size_t n_threads = n_packets > (size_t)a->sh.n_freq ? n_packets : (size_t)a->sh.n_freq;   // also zeroes lost_dev[F]
        packet_claim_kernel<<<(unsigned)((n_threads + 255) / 256), 256, 0, s>>>((const uint8_t *)packets, (unsigned)n_packets, seq0, a->sh,
                                                                               owner, a->counts, lost_dev);
        XC_CUDA(a, cudaGetLastError());
        a->launches += 1;
    }
    // grid-stride over the positions: exactly one wave of resident CTAs (256 threads each)
    unsigned blocks = (unsigned)a->n_sms * (unsigned)a->ctas_per_sm[h ? 1 : 0];
    if (blocks > a->n_positions) blocks = a->n_positions;
    if (h)
        assemble_kernel<true><<<blocks, 256, 0, s>>>((const uint8_t *)packets, a->sh, owner, owner_next, (uint8_t *)frame_dev, flags_dev,
                                                     lost_dev, a->counts, counts_dev, h->flag_x,
                                                     h->flag_cnt + (size_t)h->norm_half * h->n_freq * h->n_inputs,
                                                     h->lost_dev_acc + (size_t)h->norm_half * h->n_freq);
    else
        assemble_kernel<false><<<blocks, 256, 0, s>>>((const uint8_t *)packets, a->sh, owner, owner_next, (uint8_t *)frame_dev, flags_dev,
                                                      lost_dev, a->counts, counts_dev, nullptr, nullptr, nullptr);
    {
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) {
            // packet_claim_kernel is in the stream and has dirtied this call's table and the counters, but nothing will clean
            // them (that is assemble_kernel's job and `calls` does not advance): put the "all clean on entry" state back by
            // hand so that a later call does not read this frame's owners as its own
            a->last_cuda_error = (int)e;
            cudaMemsetAsync(a->owner, 0xFF, sizeof(uint32_t) * 2 * (size_t)a->n_positions, s);
            cudaMemsetAsync(a->counts, 0, sizeof(uint32_t) * 8, s);
            cudaGetLastError();
            return XCORR_ECUDA;
        }
    }
    a->launches += 1;
    a->calls += 1;   // the tables swap roles only once both kernels are in the stream
    if (h) {
        h->flags_dirty = true;
        h->lost_dev_dirty = true;
    }
    return XCORR_OK;
}

extern "C" int xcorr_assemble(xcorr_assembler *a, const void *packets, size_t n_packets, uint64_t seq0, void *frame_dev,
                              uint8_t *flags_dev, int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream)
{
    return assemble_common(a, nullptr, packets, n_packets, seq0, frame_dev, flags_dev, lost_dev, counts_dev, cuda_stream);
}

extern "C" int xcorr_assemble_accounted(xcorr_assembler *a, xcorr_handle *h, const void *packets, size_t n_packets, uint64_t seq0,
                                        void *frame_dev, uint8_t *flags_dev, int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream)
{
    if (!h) return XCORR_EINVAL;
    return assemble_common(a, h, packets, n_packets, seq0, frame_dev, flags_dev, lost_dev, counts_dev, cuda_stream);
}

// ---------------------------------------------------------------------------------------------------
// streamed packet path: page-locked packet ring -> H2D -> assemble -> correlate (-> flag / loss accounting)
// ---------------------------------------------------------------------------------------------------
extern "C" int xcorr_stream_attach_assembler(xcorr_stream *s, xcorr_assembler *a, size_t max_packets)
{
    if (!s || !a || max_packets == 0 || max_packets > 0x7FFFFFFEull || s->assembler) return XCORR_EINVAL;
    xcorr_handle *h = s->h;
    if (a->sh.n_inputs != h->n_inputs || a->sh.n_freq != h->n_freq || a->sh.n_time != h->n_time) return XCORR_EINVAL;
    for (int k = 0; k < s->depth; ++k) {
        if (cudaMalloc(&s->pkt_buf[k], max_packets * (size_t)a->sh.packet_bytes) != cudaSuccess) {
            h->last_cuda_error = (int)cudaGetLastError();
            return XCORR_ENOMEM;
        }
    }
    s->assembler = a;
    s->max_packets = max_packets;
    return XCORR_OK;
}

extern "C" int xcorr_stream_submit_packets(xcorr_stream *s, const void *packets_host, size_t n_packets, uint64_t seq0)
{
    if (!s || !s->assembler || (!packets_host && n_packets) || n_packets > s->max_packets) return XCORR_EINVAL;
    xcorr_handle *h = s->h;
    xcorr_assembler *a = s->assembler;
    if (h->samples_since_read + (long long)h->n_time > 16777215ll) return XCORR_EOVERFLOW;
    const int k = (int)(s->submitted % (unsigned long long)s->depth);
    if (s->submitted >= (unsigned long long)s->depth) XC_CUDA(h, cudaEventSynchronize(s->consumed[k]));   // ring back-pressure
    if (n_packets)
        XC_CUDA(h, cudaMemcpyAsync(s->pkt_buf[k], packets_host, n_packets * (size_t)a->sh.packet_bytes, cudaMemcpyHostToDevice,
                                   s->copy_stream));
    XC_CUDA(h, cudaEventRecord(s->copied[k], s->copy_stream));
    XC_CUDA(h, cudaStreamWaitEvent(s->compute_stream, s->copied[k], 0));
    // with normalisation enabled the flag / loss accounting happens inside assemble_kernel (no flag field is materialised)
    int rc = assemble_common(a, h->norm ? h : nullptr, s->pkt_buf[k], n_packets, seq0, s->buf[k], nullptr, nullptr, nullptr,
                             (void *)s->compute_stream);
    if (rc != XCORR_OK) return rc;
    rc = xcorr_process(h, s->buf[k], (void *)s->compute_stream);
    if (rc != XCORR_OK) return rc;
    XC_CUDA(h, cudaEventRecord(s->consumed[k], s->compute_stream));
    s->submitted += 1;
    return XCORR_OK;
}

extern "C" int xcorr_stream_read_normalized(xcorr_stream *s, float *vis_out, int32_t *lost_matrix_out)
{
    if (!s || !vis_out) return XCORR_EINVAL;
    const int rc = xcorr_read_normalized(s->h, vis_out, lost_matrix_out, (void *)s->compute_stream);
    if (rc != XCORR_OK) return rc;
    XC_CUDA(s->h, cudaStreamSynchronize(s->compute_stream));
    return XCORR_OK;
}

// ---------------------------------------------------------------------------------------------------
// xcorr_assemble_static: packet -> frame assembly with no allocation anywhere (include/xcorr_assemble.h)
// ---------------------------------------------------------------------------------------------------
// For callers that may not allocate (per-frame threads of a running acquisition -- a cudaMalloc would stall every
// stream of the device mid-integration, PAPER.md:49 -- and processes whose device memory belongs to another
// allocator).  The scratch that xcorr_assembler_create() gets from cudaMalloc is this array instead; it is part of the
// library's device image, so every GPU that loads the image holds these bytes until the process ends.
//
//   words [0, kStaticMaxPos)               ownership table of the frame being assembled (cleared per call)
//   words [kStaticMaxPos, 2 kStaticMaxPos) the table assemble_kernel resets for "the next frame": write-only here, since
//                                          each call clears its own table and never relies on the previous call's state
//   words [2 kStaticMaxPos, +8)            the packet counters counts[0..5] of assemble_kernel.cuh (cleared per call)
//
// One array per device, shared by all callers: calls that overlap on the GPU race on it (documented in the header).
constexpr unsigned kStaticMaxPos = XCORR_ASSEMBLE_STATIC_MAX_POSITIONS;
constexpr size_t kStaticScratchWords = 2 * (size_t)kStaticMaxPos + 64;
static_assert(kStaticScratchWords * sizeof(uint32_t) == XCORR_ASSEMBLE_STATIC_SCRATCH_BYTES, "header and array disagree");
static __device__ __align__(256) uint32_t g_static_assemble_scratch[kStaticScratchWords];

// In host code `g_static_assemble_scratch` is only a handle for the runtime's symbol table, not memory the GPU can
// reach under that address: the device address has to be asked for, per device, with that device current.
constexpr int kStaticMaxDevices = 64;
struct StaticDeviceState {
    bool ready = false;
    uint32_t *scratch = nullptr;   // device address of g_static_assemble_scratch on this device
    int n_sms = 0;
    int ctas_per_sm = 0;           // resident CTAs of assemble_kernel<false> (256 threads): the grid is one wave
};
static StaticDeviceState g_static_state[kStaticMaxDevices];
static std::mutex g_static_mutex;
static thread_local int g_static_last_cuda_error = 0;

extern "C" int xcorr_assemble_static_last_cuda_error(void) { return g_static_last_cuda_error; }

#define XC_STATIC_CUDA(expr)                              \
    do {                                                  \
        cudaError_t e_ = (expr);                          \
        if (e_ != cudaSuccess) {                          \
            cudaGetLastError();                           \
            g_static_last_cuda_error = (int)e_;           \
            return XCORR_ECUDA;                           \
        }                                                 \
    } while (0)

// Once per device, `dev` current: architecture check, SM count, occupancy, device address of the scratch array.
// None of these allocates on behalf of the caller; the symbol lookup makes the runtime load the library's device
// image onto this GPU if no kernel of it has run here yet (which is why the first call belongs to start-up).
static int static_assemble_setup(int dev, StaticDeviceState *out)
{
    std::lock_guard<std::mutex> guard(g_static_mutex);
    StaticDeviceState &st = g_static_state[dev];
    if (!st.ready) {
        int major = 0, n_sms = 0, ctas = 0;
        XC_STATIC_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return XCORR_EARCH;
        XC_STATIC_CUDA(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));
        XC_STATIC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, assemble_kernel<false>, 256, 0));
        void *addr = nullptr;
        XC_STATIC_CUDA(cudaGetSymbolAddress(&addr, g_static_assemble_scratch));
        if (!addr || n_sms < 1 || ctas < 1) { g_static_last_cuda_error = (int)cudaErrorUnknown; return XCORR_ECUDA; }
        st.scratch = static_cast<uint32_t *>(addr);
        st.n_sms = n_sms;
        st.ctas_per_sm = ctas;
        st.ready = true;
    }
    *out = st;
    return XCORR_OK;
}

extern "C" int xcorr_assemble_static(int n_inputs, int n_freq, int t_per_frame, int samples_per_packet, int freq_per_packet,
                                     const void *packets, size_t n_packets, uint64_t seq0, void *frame_dev, uint8_t *flags_dev,
                                     int32_t *lost_dev, uint32_t *counts_dev, void *cuda_stream)
{
    // the checks of xcorr_assembler_create and of xcorr_assemble, on every call: there is no handle to remember a shape
    int rc = validate_shape(n_inputs, n_freq, t_per_frame);
    if (rc != XCORR_OK) return rc;
    const int S = samples_per_packet, C = freq_per_packet;
    if (S <= 0 || C <= 0 || t_per_frame % S != 0 || n_freq % C != 0) return XCORR_EINVAL;
    if (((long long)C * n_inputs) % 128 != 0) return XCORR_EINVAL;
    if (!frame_dev || (!packets && n_packets) || n_packets > 0x7FFFFFFEull) return XCORR_EINVAL;
    if (((uintptr_t)packets & 15u) || ((uintptr_t)frame_dev & 15u) || ((uintptr_t)flags_dev & 15u) || ((uintptr_t)lost_dev & 3u) ||
        ((uintptr_t)counts_dev & 3u))
        return XCORR_EINVAL;
    AssembleShape sh = {};
    sh.n_inputs = n_inputs; sh.n_freq = n_freq; sh.n_time = t_per_frame;
    sh.s_per_packet = S; sh.c_per_packet = C;
    sh.n_streams = n_freq / C; sh.n_blocks = t_per_frame / S;
    const unsigned long long pay = (unsigned long long)S * C * n_inputs;
    sh.packet_bytes = kPacketHeaderBytes + pay + pay / 8;
    const unsigned long long n_pos64 = (unsigned long long)sh.n_streams * (unsigned long long)sh.n_blocks;
    if (n_pos64 == 0) return XCORR_EINVAL;
    if (n_pos64 > kStaticMaxPos) return XCORR_ELIMIT;   // the table is what it is: never grown, nothing allocated instead
    const unsigned n_pos = (unsigned)n_pos64;

    int dev = -1;
    XC_STATIC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return XCORR_EINVAL;
    StaticDeviceState st;
    if ((rc = static_assemble_setup(dev, &st)) != XCORR_OK) return rc;

    cudaStream_t s = (cudaStream_t)cuda_stream;
    uint32_t *owner = st.scratch;                        // this frame's claims
    uint32_t *owner_sink = st.scratch + kStaticMaxPos;   // assemble_kernel's reset of "the other table": unused here
    uint32_t *counts = st.scratch + 2 * (size_t)kStaticMaxPos;
    // the array holds whatever the last call (any shape, any caller) left there: start from "no owner" and zero counters
    XC_STATIC_CUDA(cudaMemsetAsync(owner, 0xFF, sizeof(uint32_t) * (size_t)n_pos, s));
    XC_STATIC_CUDA(cudaMemsetAsync(counts, 0, sizeof(uint32_t) * 8, s));
    {
        const size_t n_threads = n_packets > (size_t)n_freq ? n_packets : (size_t)n_freq;   // also zeroes lost_dev[F]
        packet_claim_kernel<<<(unsigned)((n_threads + 255) / 256), 256, 0, s>>>((const uint8_t *)packets, (unsigned)n_packets, seq0, sh, owner,
                                                                               counts, lost_dev);
        XC_STATIC_CUDA(cudaGetLastError());
    }
    unsigned blocks = (unsigned)st.n_sms * (unsigned)st.ctas_per_sm;
    if (blocks > n_pos) blocks = n_pos;
    assemble_kernel<false><<<blocks, 256, 0, s>>>((const uint8_t *)packets, sh, owner, owner_sink, (uint8_t *)frame_dev, flags_dev, lost_dev,
                                                  counts, counts_dev, nullptr, nullptr, nullptr);
    XC_STATIC_CUDA(cudaGetLastError());
    return XCORR_OK;
}
