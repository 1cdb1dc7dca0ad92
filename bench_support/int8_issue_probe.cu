// int8_issue_probe.cu -- measurement support, NOT part of libxcorr.so: the issue rate of the int8 tensor pipe with
// resident operands, i.e. the ceiling any kind::i8 kernel on this part can reach (SURVEY.md section 7 step 3(iii),
// "a resident-operand tcgen05.mma.kind::i8 issue-rate microbench").
//
// One CTA pair per two SMs (as xengine_kernel): one elected lane of the leader's warp 0 issues back-to-back
//     tcgen05.mma.cta_group::2.kind::i8   M = 256 (2 x 128 lanes), N = 256, K = 32, both operands MN-major SWIZZLE_128B
// from operand tiles that sit in shared memory for the whole launch -- no TMA, no unpack, no epilogue -- alternating
// between two TMEM accumulators.  int8 ops per MMA = 2 * 256 * 256 * 32.  bench.py reports the result as
// roofline.int8_issue_ceiling_tops beside the 2 x bf16 proxy.
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "../paper_1503_06189_b200/csrc/ptx.cuh"

namespace {

constexpr int kStages = 4;                 // operand buffers cycled through (A and B tile each: 64 rows x 128 B = 2 K-steps)
constexpr int kTileBytes = 64 * 128;
constexpr int kSmemBytes = kStages * 2 * kTileBytes + 1024 + 256;
constexpr int kRing = 4;                   // commit barriers: at most kRing * kBatch MMAs in flight
constexpr int kBatch = 8;

__device__ __forceinline__ uint32_t hash32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// pattern 0: zeros; 1: bytes uniform in [0, 15] (like the product's offset operands); 2: bytes uniform over all of int8
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(128, 1) int8_issue_kernel(int n_mma, int pattern)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar0 = base + kStages * 2 * kTileBytes;
    const uint32_t tmem_slot = bar0 + 8u * kRing;
    const uint32_t rank = ptx::cluster_ctarank();
    const uint32_t warp = threadIdx.x >> 5;

    for (uint32_t w = threadIdx.x; w < kStages * 2 * kTileBytes / 4; w += blockDim.x) {
        uint32_t v = hash32(w * 2654435761u + blockIdx.x * 97u + 12345u);
        v = pattern == 0 ? 0u : (pattern == 1 ? (v & 0x0F0F0F0Fu) : v);
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(base + 4u * w), "r"(v) : "memory");
    }
    if (threadIdx.x == 0) {
        for (int k = 0; k < kRing; ++k) ptx::mbar_init(bar0 + 8u * k, 1);
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<2>(tmem_slot, 512);
        ptx::tmem_relinquish<2>();
    }
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync();
    ptx::tc_fence_after_sync();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    if (rank == 0 && warp == 0) {
        // the whole warp walks the loop and one elected lane issues, with warp-uniform descriptors (ring base + constants),
        // exactly as xengine_kernel does: issued from a divergent single-lane branch ptxas wraps every tcgen05.mma in an
        // elect / broadcast / retry loop and the issue thread, not the tensor pipe, sets the pace
        constexpr uint32_t idesc = ptx::make_idesc_i8_mnmajor(256, 256);
        const bool leader_lane = ptx::elect_one();
        const uint64_t desc0 = ptx::make_smem_desc_mn_sw128(base, 1024, 1024);
        const uint32_t desc_hi = (uint32_t)(desc0 >> 32);
        int batch = 0;
        uint32_t st = 0;                                                             // one stage = 2 K-steps of 32 rows
        for (int i = 0; i < n_mma; i += 2) {
            if (leader_lane) {
                const uint32_t lo = (uint32_t)desc0 + st * (uint32_t)((2 * kTileBytes) >> 4);
#pragma unroll
                for (uint32_t k = 0; k < 2; ++k) {
                    const uint64_t da = ptx::pack_u64(lo + k * ((32u * 128u) >> 4), desc_hi);
                    const uint64_t db = ptx::pack_u64(lo + (uint32_t)(kTileBytes >> 4) + k * ((32u * 128u) >> 4), desc_hi);
                    ptx::mma_i8<2>(tmem_base + (k ? 256u : 0u), da, db, idesc, i >= 2 ? 1u : 0u);
                }
            }
            if (++st == (uint32_t)kStages) st = 0;
            if ((i + 2) % kBatch == 0) {
                const int slot = batch % kRing;
                if (leader_lane) ptx::mma_commit<2>(bar0 + 8u * slot, 0x1);
                ++batch;
                if (batch >= kRing) {                                               // wait for the batch issued kRing - 1 batches ago
                    const int wb = batch - (kRing - 1) - 1;
                    ptx::mbar_wait(bar0 + 8u * (wb % kRing), (uint32_t)(wb / kRing) & 1u);
                }
            }
        }
        // drain: one more commit behind everything issued
        const int slot = batch % kRing;
        if (leader_lane) ptx::mma_commit<2>(bar0 + 8u * slot, 0x1);
        for (int wb = (batch >= kRing - 1 ? batch - (kRing - 1) : 0); wb <= batch; ++wb)
            ptx::mbar_wait(bar0 + 8u * (wb % kRing), (uint32_t)(wb / kRing) & 1u);
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync();
    if (warp == 1) {
        ptx::tc_fence_after_sync();
        ptx::tmem_dealloc<2>(tmem_base, 512);
    }
}

}  // namespace

// Launch the probe on the current device (must be compute capability 10.x): `launches` launches back to back, each with
// one CTA pair per two SMs issuing `mma_per_pair` MMAs; the elapsed time between CUDA events around them goes to *ms_out,
// the int8 TOP/s (2 * 256 * 256 * 32 ops per MMA) to *tops_out.  Returns 0 or a negative code (-1 bad argument,
// -2 wrong architecture, -4 CUDA error).
extern "C" int xcorr_probe_int8_issue(int mma_per_pair, int launches, int pattern, double *tops_out, double *ms_out)
{
    if (mma_per_pair <= 0 || launches <= 0 || pattern < 0 || pattern > 2 || !tops_out || !ms_out) return -1;
    if (mma_per_pair % kBatch != 0) return -1;   // the issue loop commits every kBatch MMAs
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return -4;
    if (prop.major != 10) return -2;
    const int pairs = prop.multiProcessorCount / 2;
    if (cudaFuncSetAttribute(int8_issue_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes) != cudaSuccess) return -4;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -4;
    int8_issue_kernel<<<2 * pairs, 128, kSmemBytes>>>(mma_per_pair, pattern);   // warm-up
    cudaEventRecord(e0);
    for (int k = 0; k < launches; ++k) int8_issue_kernel<<<2 * pairs, 128, kSmemBytes>>>(mma_per_pair, pattern);
    cudaEventRecord(e1);
    const cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return -4;
    const double ops = 2.0 * 256.0 * 256.0 * 32.0 * (double)mma_per_pair * (double)pairs * (double)launches;
    *ms_out = ms;
    *tops_out = ops / (ms * 1e-3) / 1e12;
    return 0;
}
