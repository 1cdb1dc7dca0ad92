// xengine_kernel.cuh -- the fused X-engine kernel for sm_100a (hot-path rows a1..a4).
//
//   a1  TMA stages packed bytes  frame[t][f][128 inputs]  as 128-byte rows (SWIZZLE_128B) into smem, kPackedStages deep
//   a2  unpack warps split each byte into int8 planes (same swizzled 128-byte-row layout, so the unpack is purely
//       element-wise and never looks at the swizzle).  The planes hold the OFFSET values h' = Re + 8, l' = Im + 8 in
//       [0, 15] and, per tile kind, s' = h' + l' or the complement 15 - l' (layout.hpp "OFFSET OPERANDS": constant-zero
//       upper bits cut the MMA datapath's switching power, and the part is power-limited); the same warps keep per-input
//       column sums of h', l' so that xcorr_read can remove the offsets exactly.  The 8 unpack warps work in groups on
//       alternate stages (KernelCfg::kUnpackGroups)
//   a3  one elected lane of the MMA warp issues 2-CTA tcgen05.mma kind::i8 (M = 256 over the CTA pair, N = 256, K = 32)
//       with both operands MN-major straight from those planes, every operand warp-uniform; int32 accumulators stay in
//       TMEM (512 columns) for the whole time range of the work segment
//   a4  epilogue warps tcgen05.ld the accumulators and write them into this segment's accumulator slot: 16-byte stores
//       (first frame of an integration) or, through a shared-memory staging buffer, bulk reduce-adds (later frames)
//
// Complex product from real GEMMs (BASELINE.json:north_star (b)); h = Re plane, l = Im plane, s = h + l (offset values):
//   off-diagonal        (I <  J):   R += h_I h_J^T ; Q += l_I h_J^T ; R += l_I l_J^T ; Q += h_I (15 - l_J)^T     (4 MMAs per K-step)
//   diagonal super-tile (I == J):   R += s s^T ; Q += l h^T                                                     (2 MMAs per K-step)
// On the diagonal the tile is Hermitian, which lets three real products per complex MAC do (Gauss), two of them being the
// two triangles of ONE full product:  with G = (h+l)(h+l)^T = hh^T + ll^T + hl^T + lh^T (symmetric) and X = l h^T,
//     Re V[i,j] = G[i,j] - X[i,j] - X[j,i]        Im V[i,j] = X[i,j] - X[j,i]        (formed by xcorr_read, exact, no division)
// so a diagonal super-tile costs 2 x 256 x 256 MACs per sample where the stacked form (hh^T, ll^T, lh^T) costs 3 -- at
// N = 256 (every tile is diagonal) the kernel issues 0.996 of the "useful" 4 real MACs per complex pair i <= j.
// Integer MMAs have no operand-negate bit, hence the explicit complement plane 15 - l'_J for I < J (the constant
// 15 sum h'_I it adds is removed at read together with the offsets).
//
// One cluster = CTA pair = one "worker" of schedule.hpp; CTA rank r owns inputs [128r, 128r+128) of the
// row super-block (A operand, TMEM lanes) and of the column super-block (its half of the B operand).
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "layout.hpp"
#include "ptx.cuh"
#include "schedule.hpp"

namespace xc {

// ------------------------------------------------------------------------------------------------
// compile-time configuration
// ------------------------------------------------------------------------------------------------
template <bool kOffDiag>
struct KernelCfg {
    static constexpr int kRowBytes = 128;                          // one t-row of one 128-input block
    static constexpr int kPlaneBytes = kStageT * kRowBytes;        // 8 KiB: one plane (or packed block) per stage
    static constexpr int kPackedBlocks = kOffDiag ? 2 : 1;         // A block (+ B block when I < J)
    static constexpr int kPlanes = kOffDiag ? 5 : 3;               // h_a l_a s_a   or   h_a l_a {s_a | h_b} l_b 15-l_b
    static constexpr int kPackedStageBytes = kPackedBlocks * kPlaneBytes;
    static constexpr int kPlaneStageBytes = kPlanes * kPlaneBytes;
    static constexpr int kPackedStages = kOffDiag ? 4 : 8;
    static constexpr int kPlaneStages = kOffDiag ? 3 : 5;
    static constexpr int kUnpackWarps = 8;                         // multiple of 4
    static constexpr int kUnpackThreads = kUnpackWarps * 32;
    static constexpr int kWarpEpi0 = 4 + kUnpackWarps;             // epilogue warps: warp % 4 == TMEM lane quarter
    static constexpr int kThreads = (4 + kUnpackWarps + 4) * 32;
    static constexpr int kSumPlanes = 2 * kPackedBlocks;           // column sums kept by the unpack warps: h'_a l'_a [h'_b l'_b]
    static constexpr int kSumScratch = kUnpackThreads * 32;        // cross-thread reduction of the column sums (8 KiB)
    static constexpr int kEpiStageBytes = 32 * 32 * 4;             // one chunk of a warp: 32 rows x 32 columns int32 = 4 KiB
    static constexpr int kEpiStaging = 4 * 2 * kEpiStageBytes;     // 4 epilogue warps x 2 buffers (32 KiB)
    static constexpr int kSmemData = kPackedStages * kPackedStageBytes + kPlaneStages * kPlaneStageBytes + kSumScratch + kEpiStaging;
    static constexpr int kSmemBytes = kSmemData + 1024 /*align slack*/ + 1024 /*barriers*/;
    // The unpack warps work in kUnpackGroups groups; group g takes the stages it == g (mod kUnpackGroups), so several stages
    // are unpacked at the same time and a warp's per-stage chain (barrier waits -> ld.shared -> ALU -> st.shared -> proxy
    // fence -> arrive) is paid once per kUnpackGroups stages: with one group that chain (about 630 clk per stage) was what
    // bounded the kernel once the diagonal tiles dropped to 2 MMAs per K-step.
    static constexpr int kUnpackGroups = kOffDiag ? 2 : 4;
    static constexpr int kGroupWarps = kUnpackWarps / kUnpackGroups;
    static constexpr int kGroupThreads = kGroupWarps * 32;
    // column sums: a thread sees kRowsPerStage rows of its 16 inputs per stage it unpacks; byte lanes hold 17 rows of values
    // <= 15, 16-bit lanes 4369 rows
    static constexpr int kRowsPerStage = kPlaneBytes / (kGroupThreads * 16);
    static constexpr int kLoadBatch = 4;                                        // rows (16-byte loads) a thread has in flight at a time
    static constexpr int kWidenStages = 16 / kRowsPerStage;                     // in stages of the thread's own group
    static constexpr int kFlushEpoch = 1024;                                    // in stages of the segment (all groups): 2048 rows per thread
    static_assert(kUnpackThreads == 256, "the column-sum reduction assumes 256 unpack threads (32 rows x 8 chunks per pass)");
    static_assert(kGroupThreads % 64 == 0, "a thread must keep the same 16 inputs: rows per pass must be a multiple of 8");
    static_assert(kRowsPerStage >= 1 && kRowsPerStage <= 16 && 16 % kRowsPerStage == 0, "stage size vs column-sum lanes");
    static_assert(kRowsPerStage % kLoadBatch == 0, "rows per stage vs load batch");
    static_assert(kFlushEpoch / kUnpackGroups * kRowsPerStage <= 4096, "16-bit column-sum lanes");
    // mbarrier waits are by phase PARITY, which is only sound while a waiter can never be two phases ahead of the barrier.
    // Packed ring (TMA -> unpack): the loads of different stages may land out of order, so a slot must always be consumed
    // by the same group -- kPackedStages is a multiple of kUnpackGroups (with 3 slots and 2 groups a group could reach its
    // next use of a slot while the other group's load into that slot was still in flight, pass the wait on the stale
    // parity and unpack old bytes: seen as wrong visibilities on C5).  Plane ring (unpack -> MMA -> unpack): its phases
    // complete through tcgen05.commit, in issue order.  A group at stage `it` waits for commit(it - ring) and would pass
    // wrongly only if commit(it - 2 ring) were still outstanding; at its previous stage it - groups it waited for
    // commit(it - groups - ring), which is at or after commit(it - 2 ring) whenever ring >= groups -- so any ring size not
    // smaller than the group count is sound there, multiples or not.
    static_assert(kPackedStages % kUnpackGroups == 0, "a packed slot must always be consumed by the same unpack group");
    static_assert(kPlaneStages >= kUnpackGroups, "plane ring: a group's previous wait must cover the phase before the one it waits for");
};

constexpr int kWarpTma = 0;
constexpr int kWarpMma = 1;
constexpr int kWarpTmem = 2;
constexpr int kWarpUnpack0 = 4;        // unpack warps 4 .. 4 + Cfg::kUnpackWarps - 1, then 4 epilogue warps
constexpr int kNumEpiWarps = 4;

constexpr int kMaxHeadWorkers = 80;   // workers whose first segment also travels in the kernel parameters (74 on a B200)

struct KernelParams {
    // every worker's FIRST segment, in the parameter (constant) bank: the schedule tables below are evicted from L2 by every
    // frame that streams through, and two dependent cold loads (worker_begin -> segments) kept the first frame load back by
    // about 2 k clk.  A worker without segments has stage_begin == stage_end here.
    Segment head[kMaxHeadWorkers];
    const Segment *segments;       // device
    const int32_t *worker_begin;   // device, n_workers + 1
    int32_t *acc;                  // device accumulator slots, layout.hpp
    int32_t *sums;                 // device column-sum slots, layout.hpp
    int first_frame;               // 1: first frame of an integration -> epilogue stores; 0: load-add-store
    int n_inputs;
    int n_freq;
    int n_time;
    int wait_frame;                // 1: the TMA lane waits for the previous kernel of the stream before the first frame load
};

// ------------------------------------------------------------------------------------------------
// a2: nibble unpack, 4 samples per 32-bit word, to OFFSET values x' = sext4(nibble) + 8 = nibble ^ 8  (R2, R3)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t unpack_re4(uint32_t w) { return ((w >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u; }   // h' = Re + 8
__device__ __forceinline__ uint32_t unpack_im4(uint32_t w) { return (w & 0x0F0F0F0Fu) ^ 0x08080808u; }          // l' = Im + 8
__device__ __forceinline__ uint32_t complement4(uint32_t y) { return y ^ 0x0F0F0F0Fu; }                          // 15 - y per byte

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
template <bool kOffDiag>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(KernelCfg<kOffDiag>::kThreads, 1)
xengine_kernel(const __grid_constant__ CUtensorMap frame_map, const KernelParams p)
{
    using Cfg = KernelCfg<kOffDiag>;
    extern __shared__ uint8_t smem_raw[];

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();          // 0 = leader (issues the MMAs)
    const uint32_t worker = blockIdx.x >> 1;

    // ---- shared memory carve-up (1024-byte aligned data, then barriers) ----
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t smem_packed = smem_base;
    const uint32_t smem_planes = smem_packed + Cfg::kPackedStages * Cfg::kPackedStageBytes;
    const uint32_t smem_sumscratch = smem_planes + Cfg::kPlaneStages * Cfg::kPlaneStageBytes;
    const uint32_t smem_epistage = smem_sumscratch + Cfg::kSumScratch;
    const uint32_t bar_base = smem_epistage + Cfg::kEpiStaging;
    // barrier slots (8 bytes each)
    auto bar_pk_full = [&](int s) { return bar_base + 8u * (uint32_t)s; };
    auto bar_pk_empty = [&](int s) { return bar_base + 8u * (uint32_t)(Cfg::kPackedStages + s); };
    auto bar_pl_full = [&](int s) { return bar_base + 8u * (uint32_t)(2 * Cfg::kPackedStages + s); };
    auto bar_pl_empty = [&](int s) { return bar_base + 8u * (uint32_t)(2 * Cfg::kPackedStages + Cfg::kPlaneStages + s); };
    const uint32_t bar_acc_full = bar_base + 8u * (uint32_t)(2 * Cfg::kPackedStages + 2 * Cfg::kPlaneStages);
    const uint32_t bar_acc_empty = bar_acc_full + 8u;
    const uint32_t tmem_slot = bar_acc_empty + 8u;   // uint32 written by tcgen05.alloc

    // PDL: the next kernel of the stream may begin its own prologue; it waits (grid_dependency_wait) for this grid's completion
    ptx::grid_launch_dependents();

    const int seg_begin = p.worker_begin[worker];          // static schedule tables: not written by any kernel
    const int seg_end = p.worker_begin[worker + 1];

    // N <= 256: every frame byte is read exactly once -> evict-first in L2, so the accumulator slots written by the
    // epilogue are still there when xcorr_read's finalize pass wants them (C2 step 122.3 -> 119.7 us; less HBM traffic
    // also means less power, and the part is power-limited).  For N > 256 the blocks are re-read by the neighbouring
    // super-tiles through L2 and keep the default policy.
    const uint64_t frame_policy = ptx::l2_policy_evict_first();
    // a1 issues one packed stage: one box (two when I < J) of kStageT rows x 128 inputs, 128-byte swizzle
    auto tma_issue = [&](const Segment &seg, int st, uint32_t slot) {
        const uint32_t dst = smem_packed + slot * Cfg::kPackedStageBytes;
        const bool off = kOffDiag && (seg.I != seg.J);
        ptx::mbar_arrive_expect_tx(bar_pk_full(slot), off ? 2 * Cfg::kPlaneBytes : Cfg::kPlaneBytes);
        if constexpr (!kOffDiag) {
            ptx::tma_load_3d_hint(dst, &frame_map, bar_pk_full(slot), seg.I * kSuper + (int)rank * kBlock, seg.f, st * kStageT, frame_policy);
            return;
        }
        ptx::tma_load_3d(dst, &frame_map, bar_pk_full(slot), seg.I * kSuper + (int)rank * kBlock, seg.f, st * kStageT);
        if (off)
            ptx::tma_load_3d(dst + Cfg::kPlaneBytes, &frame_map, bar_pk_full(slot), seg.J * kSuper + (int)rank * kBlock, seg.f, st * kStageT);
    };
    uint32_t tma_pre = 0;   // packed stages the TMA lane put in flight before the prologue barrier (their slots start empty)

    if (warp == kWarpMma && lane == 0) {
        for (int s = 0; s < Cfg::kPlaneStages; ++s) {
            ptx::mbar_init(bar_pl_full(s), 2 * Cfg::kGroupWarps);   // the unpack warps of one group, BOTH CTAs (used in the leader only)
            ptx::mbar_init(bar_pl_empty(s), 1);                   // tcgen05.commit (multicast to both CTAs)
        }
        ptx::mbar_init(bar_acc_full, 1);                          // tcgen05.commit (multicast)
        ptx::mbar_init(bar_acc_empty, 2 * kNumEpiWarps);          // epilogue warps of BOTH CTAs (leader only)
        ptx::fence_mbar_init();
    }
    // the TMA warp walks its loops as a whole and one elected lane issues (warp-uniform operands: see the MMA issuer)
    bool tma_leader = false;
    if (warp == kWarpTma) {
        tma_leader = ptx::elect_one();
        if (tma_leader) {
            ptx::prefetch_tensormap(&frame_map);
            for (int s = 0; s < Cfg::kPackedStages; ++s) {
                ptx::mbar_init(bar_pk_full(s), 1);                    // TMA producer's arrive.expect_tx
                ptx::mbar_init(bar_pk_empty(s), Cfg::kGroupWarps);      // one arrive per unpack warp of the stage's group
            }
            ptx::fence_mbar_init();
            ptx::fence_proxy_async_smem();
        }
        __syncwarp();
        // the packed barriers and slots are this CTA's own: start the first loads now, so the frame is already on its
        // way while TMEM is allocated and the cluster synchronises
        // the frame may be the output of the previous kernel of the stream, which may have let this grid start early:
        // wait for it, unless the caller has promised complete frames (xcorr_promise_complete_frames)
        if (p.wait_frame) ptx::grid_dependency_wait();
        // (the first segment's stages only: its description comes with the kernel parameters, see KernelParams::head)
        if (worker < (uint32_t)kMaxHeadWorkers) {
            const Segment seg = p.head[worker];
            for (int st = seg.stage_begin; st < seg.stage_end && tma_pre < (uint32_t)Cfg::kPackedStages; ++st, ++tma_pre)
                if (tma_leader) tma_issue(seg, st, tma_pre);
        }
    }
    if (warp == kWarpTmem) {
        ptx::tmem_alloc<2>(tmem_slot, kAccCols);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    // barriers of both CTAs initialised before any remote arrive / multicast commit.  The arrive is RELAXED: the barrier
    // initialisations were published by fence.mbarrier_init.release.cluster, and a releasing arrive would make every thread
    // wait here for the frame loads already in flight (measured: 3.5-4 k clk per CTA)
    ptx::cluster_arrive_relaxed();
    ptx::cluster_wait();
    ptx::tc_fence_after_sync();
    // The accumulator / sum slots may still be read or written by the previous kernel of the stream (xcorr_read's
    // finalize_kernel, or the previous frame's xengine_kernel): the warps that touch them wait (griddepcontrol.wait) right
    // before their first access -- the unpack warps before a segment's column sums go out, the epilogue warps before the
    // first chunk -- so loading, unpacking and multiplying the first segment overlap the previous kernel's tail.

    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    if (warp == kWarpTma) {
        // ===================================================== a1: TMA producer (whole warp, one elected lane issues)
        {
            uint32_t it = 0, slot = 0, ph = 0;
            for (int sg = seg_begin; sg < seg_end; ++sg) {
                const Segment seg = p.segments[sg];
                for (int st = seg.stage_begin; st < seg.stage_end; ++st, ++it) {
                    if (it >= tma_pre) {                           // (the first tma_pre stages are in flight since the prologue)
                        ptx::mbar_wait(bar_pk_empty(slot), ph ^ 1u);
                        if (tma_leader) tma_issue(seg, st, slot);
                    }
                    if (++slot == (uint32_t)Cfg::kPackedStages) { slot = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == kWarpMma) {
        // ===================================================== a3: MMA issuer (leader CTA; the whole warp walks the loop, one
        // elected lane issues).  Every value the tcgen05 instructions take is warp-uniform and kept so: the ring position and
        // phase are carried incrementally, a descriptor is the ring base's low word plus small constants (ptx::make_smem_desc
        // layout: address >> 4 in the low bits).  Issued from a divergent single-lane branch instead, ptxas wraps every MMA in
        // an elect / broadcast / retry loop (about 30 instructions per MMA) and the issue thread, not the tensor pipe, sets
        // the pace: 155 clk per MMA against 128.
        if (rank == 0) {
            constexpr uint32_t idesc = ptx::make_idesc_i8_mnmajor(256, 256);
            constexpr uint32_t kDescPlane = Cfg::kPlaneBytes >> 4;                  // + one plane
            constexpr uint32_t kDescK = (32u * Cfg::kRowBytes) >> 4;               // + one K-step of 32 rows
            const bool leader_lane = ptx::elect_one();
            const uint32_t tmem_R = tmem_base;
            const uint32_t tmem_Q = tmem_base + 256;
            const uint64_t desc0 = ptx::make_smem_desc_mn_sw128(smem_planes, 1024, 1024);   // plane 0 of ring slot 0
            const uint32_t desc_hi = (uint32_t)(desc0 >> 32);
            uint32_t slot = 0, ph = 0, unit = 0;
            for (int sg = seg_begin; sg < seg_end; ++sg, ++unit) {
                const Segment seg = p.segments[sg];
                const bool off = kOffDiag && (seg.I != seg.J);
                ptx::mbar_wait_cluster(bar_acc_empty, (unit & 1u) ^ 1u);     // epilogues of both CTAs drained TMEM
                ptx::tc_fence_after_sync();
                for (int st = seg.stage_begin; st < seg.stage_end; ++st) {
                    ptx::mbar_wait_cluster(bar_pl_full(slot), ph);
                    ptx::tc_fence_after_sync();
                    if (leader_lane) {
                        const uint32_t lo = (uint32_t)desc0 + slot * (uint32_t)(Cfg::kPlaneStageBytes >> 4);
                        auto desc = [&](uint32_t plane, uint32_t k) { return ptx::pack_u64(lo + plane * kDescPlane + k * kDescK, desc_hi); };
#pragma unroll
                        for (uint32_t k = 0; k < (uint32_t)kStageT / 32u; ++k) {
                            const uint32_t acc = (st != seg.stage_begin || k != 0) ? 1u : 0u;
                            if (!off) {
                                ptx::mma_i8<2>(tmem_R, desc(2, k), desc(2, k), idesc, acc);   // R (= G) = s s^T,  s = h + l
                                ptx::mma_i8<2>(tmem_Q, desc(1, k), desc(0, k), idesc, acc);   // Q (= X) = l h^T
                            } else {
                                ptx::mma_i8<2>(tmem_R, desc(0, k), desc(2, k), idesc, acc);   // R  = h_I h_J^T
                                ptx::mma_i8<2>(tmem_Q, desc(1, k), desc(2, k), idesc, acc);   // Q  = l_I h_J^T
                                ptx::mma_i8<2>(tmem_R, desc(1, k), desc(3, k), idesc, 1u);    // R += l_I l_J^T
                                ptx::mma_i8<2>(tmem_Q, desc(0, k), desc(4, k), idesc, 1u);    // Q += h_I (-l_J)^T
                            }
                        }
                        ptx::mma_commit<2>(bar_pl_empty(slot), 0x3);   // planes of this stage may be overwritten (both CTAs)
                    }
                    if (++slot == (uint32_t)Cfg::kPlaneStages) { slot = 0; ph ^= 1u; }
                }
                if (leader_lane) ptx::mma_commit<2>(bar_acc_full, 0x3);             // accumulators complete (both CTAs)
            }
        }
    } else if (warp >= kWarpUnpack0 && warp < (uint32_t)Cfg::kWarpEpi0) {
        // ===================================================== a2: unpack warps
        // A group of kGroupThreads threads unpacks a stage; thread `gtid` of the group handles the 16-byte chunks at byte offsets
        // (q * kGroupThreads + gtid) * 16 of every 8 KiB block: row q * kGroupThreads / 8 + gtid / 8, chunk position gtid % 8.
        // TMA's 128-byte swizzle puts logical chunk c of row k at position c ^ (k % 8), so the thread always sees the same 16
        // inputs  [16 c_t, 16 c_t + 16),  c_t = (tid % 8) ^ ((tid / 8) % 8)  -- which is what lets it keep their column sums in
        // registers: byte lanes (<= 16 rows), widened to 16-bit lanes (<= 4096 rows), reduced over the 32 threads that share
        // a chunk through smem into an int32 total held by thread `input index` (< 128).
        const uint32_t tid = threadIdx.x - kWarpUnpack0 * 32;     // 0 .. 255
        const uint32_t group = tid / Cfg::kGroupThreads;
        const uint32_t gtid = tid % Cfg::kGroupThreads;
        const uint32_t pl_full_leader = ptx::mapa(bar_base, 0) + (bar_pl_full(0) - bar_base);
        uint32_t bsum[Cfg::kSumPlanes][4];    // byte lanes   : word k = inputs 4k .. 4k+3 of the chunk
        uint32_t wsum[Cfg::kSumPlanes][8];    // 16-bit lanes : [k] = bytes 0, 2 of word k ; [4 + k] = bytes 1, 3
        uint32_t tot[Cfg::kSumPlanes];        // tid < 128: int32 column sum of input `tid` of the block, this segment so far
#pragma unroll
        for (int pl = 0; pl < Cfg::kSumPlanes; ++pl) {
            tot[pl] = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) bsum[pl][k] = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) wsum[pl][k] = 0;
        }
        auto widen = [&]() {
#pragma unroll
            for (int pl = 0; pl < Cfg::kSumPlanes; ++pl)
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    wsum[pl][k] += bsum[pl][k] & 0x00FF00FFu;
                    wsum[pl][4 + k] += (bsum[pl][k] >> 8) & 0x00FF00FFu;
                    bsum[pl][k] = 0;
                }
        };
        // where thread `tid` (< 128, input index inside the block) finds its input in a contributor's 32-byte record
        const uint32_t red_chunk = tid >> 4;
        const uint32_t red_off = ((((tid & 1u) << 2) + ((tid & 15u) >> 2)) << 2) + (((tid & 3u) >> 1) << 1);
        auto flush = [&](int n_planes) {
            widen();
#pragma unroll
            for (int pl = 0; pl < Cfg::kSumPlanes; ++pl) {
                if (pl < n_planes) {
                    const uint32_t rec = smem_sumscratch + tid * 32u;
                    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(rec), "r"(wsum[pl][0]), "r"(wsum[pl][1]), "r"(wsum[pl][2]),
                                 "r"(wsum[pl][3])
                                 : "memory");
                    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(rec + 16u), "r"(wsum[pl][4]), "r"(wsum[pl][5]),
                                 "r"(wsum[pl][6]), "r"(wsum[pl][7])
                                 : "memory");
                    asm volatile("bar.sync 1, 256;" ::: "memory");
                    if (tid < 128) {
                        uint32_t acc = 0;
#pragma unroll 8
                        for (uint32_t row = 0; row < 32; ++row) {
                            const uint32_t contributor = 8u * row + (red_chunk ^ (row & 7u));
                            uint32_t v;
                            asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(smem_sumscratch + contributor * 32u + red_off));
                            acc += v;
                        }
                        tot[pl] += acc;
                    }
                    asm volatile("bar.sync 1, 256;" ::: "memory");
#pragma unroll
                    for (int k = 0; k < 8; ++k) wsum[pl][k] = 0;
                }
            }
        };
        // one 8 KiB packed block -> its planes, kLoadBatch rows at a time: the batch's loads first, then unpack / sum / store
        auto load_batch = [&](uint32_t src, int q0, uint32_t (&w)[Cfg::kLoadBatch][4]) {
#pragma unroll
            for (int q = 0; q < Cfg::kLoadBatch; ++q)
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                             : "=r"(w[q][0]), "=r"(w[q][1]), "=r"(w[q][2]), "=r"(w[q][3])
                             : "r"(src + (uint32_t)((q0 + q) * Cfg::kGroupThreads + gtid) * 16u));
        };
        auto st_v4 = [&](uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
            asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
        };
        uint32_t it = 0;
        for (int sg = seg_begin; sg < seg_end; ++sg) {
            const Segment seg = p.segments[sg];
            const bool off = kOffDiag && (seg.I != seg.J);
            int since_widen = 0, epochs_done = 0;
            for (int st = seg.stage_begin; st < seg.stage_end; ++st, ++it) {
                if (it % Cfg::kUnpackGroups != group) continue;               // another group's stage
                // 16-bit lanes: every thread joins a flush per kFlushEpoch stages of the segment (the same number in every group)
                for (; epochs_done < (st - seg.stage_begin) / Cfg::kFlushEpoch; ++epochs_done) { flush(off ? 4 : 2); since_widen = 0; }
                const uint32_t pslot = it % Cfg::kPackedStages, pph = (it / Cfg::kPackedStages) & 1u;
                const uint32_t lslot = it % Cfg::kPlaneStages, lph = (it / Cfg::kPlaneStages) & 1u;
                ptx::mbar_wait(bar_pk_full(pslot), pph);                      // TMA bytes landed
                const uint32_t src = smem_packed + pslot * Cfg::kPackedStageBytes;
                const uint32_t dst = smem_planes + lslot * Cfg::kPlaneStageBytes;
                uint32_t w[Cfg::kLoadBatch][4];
                load_batch(src, 0, w);
                ptx::mbar_wait_cluster(bar_pl_empty(lslot), lph ^ 1u);        // MMAs that read this plane slot retired
#pragma unroll
                for (int q0 = 0; q0 < Cfg::kRowsPerStage; q0 += Cfg::kLoadBatch) {
                    if (q0 > 0) load_batch(src, q0, w);
#pragma unroll
                    for (int q = 0; q < Cfg::kLoadBatch; ++q) {
                        const uint32_t o = (uint32_t)((q0 + q) * Cfg::kGroupThreads + gtid) * 16u;
                        uint32_t re[4], im[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            re[k] = unpack_re4(w[q][k]);
                            im[k] = unpack_im4(w[q][k]);
                            bsum[0][k] += re[k];
                            bsum[1][k] += im[k];
                        }
                        st_v4(dst + o, re[0], re[1], re[2], re[3]);
                        st_v4(dst + Cfg::kPlaneBytes + o, im[0], im[1], im[2], im[3]);
                        if (!off)   // diagonal super-tile: s' = h' + l' in [0, 30] per byte (no carries between bytes)
                            st_v4(dst + 2 * Cfg::kPlaneBytes + o, re[0] + im[0], re[1] + im[1], re[2] + im[2], re[3] + im[3]);
                    }
                }
                if constexpr (kOffDiag) {
                    if (off) {
#pragma unroll
                        for (int q0 = 0; q0 < Cfg::kRowsPerStage; q0 += Cfg::kLoadBatch) {
                            load_batch(src + Cfg::kPlaneBytes, q0, w);
#pragma unroll
                            for (int q = 0; q < Cfg::kLoadBatch; ++q) {
                                const uint32_t o = (uint32_t)((q0 + q) * Cfg::kGroupThreads + gtid) * 16u;
                                uint32_t re[4], im[4];
#pragma unroll
                                for (int k = 0; k < 4; ++k) {
                                    re[k] = unpack_re4(w[q][k]);
                                    im[k] = unpack_im4(w[q][k]);
                                    bsum[Cfg::kSumPlanes - 2][k] += re[k];
                                    bsum[Cfg::kSumPlanes - 1][k] += im[k];
                                }
                                st_v4(dst + 2 * Cfg::kPlaneBytes + o, re[0], re[1], re[2], re[3]);
                                st_v4(dst + 3 * Cfg::kPlaneBytes + o, im[0], im[1], im[2], im[3]);
                                st_v4(dst + 4 * Cfg::kPlaneBytes + o, complement4(im[0]), complement4(im[1]), complement4(im[2]), complement4(im[3]));
                            }
                        }
                    }
                }
                ptx::fence_proxy_async_smem();       // my plane writes -> visible to the tensor core's smem reads
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive_local(bar_pk_empty(pslot));                       // packed slot may be refilled
                    ptx::mbar_arrive_cluster(pl_full_leader + 8u * lslot);             // tell the leader's MMA thread
                }
                if (++since_widen == Cfg::kWidenStages) { widen(); since_widen = 0; }
            }
            for (; epochs_done < (seg.stage_end - seg.stage_begin - 1) / Cfg::kFlushEpoch; ++epochs_done) flush(off ? 4 : 2);
            // segment done: this segment's column sums -> its sum slot (same store / load-add-store rule as the epilogue)
            ptx::grid_dependency_wait();                           // sum slots: see the note at the prologue
            flush(off ? 4 : 2);
            if (tid < 128) {
                int32_t *dst_sum = p.sums + ((size_t)seg.slot * 2 + rank) * (size_t)kSumElemsPerCta + tid;
#pragma unroll
                for (int pl = 0; pl < Cfg::kSumPlanes; ++pl) {
                    if (pl < (off ? 4 : 2)) {
                        const int32_t old = p.first_frame ? 0 : dst_sum[pl * kBlock];
                        dst_sum[pl * kBlock] = old + (int32_t)tot[pl];
                    }
                    tot[pl] = 0;
                }
            }
        }
    } else if (warp >= (uint32_t)Cfg::kWarpEpi0) {
        // ===================================================== a4: epilogue warps
        const uint32_t quarter = warp & 3u;                      // TMEM lanes [32*quarter, 32*quarter+32)
        const uint32_t acc_empty_leader = ptx::mapa(bar_acc_empty, 0);
        uint32_t unit = 0;
        uint32_t epi_chunks = 0;                                 // chunks this warp has handed to the bulk engine so far
        for (int sg = seg_begin; sg < seg_end; ++sg, ++unit) {
            const Segment seg = p.segments[sg];
            ptx::mbar_wait_cluster(bar_acc_full, unit & 1u);
            ptx::tc_fence_after_sync();
            ptx::grid_dependency_wait();                           // accumulator slots: see the note at the prologue
            const int row0 = (int)(rank * kBlock + quarter * 32);             // first row of this warp inside the super-block
            const int rows_valid = p.n_inputs - seg.I * kSuper - row0;         // rows of this warp that are real inputs
            const int cols_valid = min(kSuper, p.n_inputs - seg.J * kSuper);   // columns that are real inputs
            // this warp's 64 KiB of the segment's own slot: [col / 4][row % 32][4] int32, columns contiguous -> one warp's 16-byte
            // accesses are 512 B contiguous
            int32_t *slot_warp = p.acc + ((size_t)seg.slot * 2 + rank) * (size_t)kAccElemsPerCta + (size_t)quarter * kAccElemsPerQuarter;
            // this warp's last TMEM load has landed: the next unit's MMAs may overwrite the accumulators
            bool released = false;
            auto release_tmem = [&]() {
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(acc_empty_leader);
                released = true;
            };
            if (rows_valid > 0) {
                // R columns.  On a diagonal super-tile R (= G) is symmetric and only j >= i is wanted: a warp starts at its first
                // row, and the 128 x 128 block G[0:128, 128:256] -- held by CTA 0 as is and by CTA 1 transposed -- is SHARED between
                // the two CTAs: CTA 0 writes its columns 128..191, CTA 1 writes the rest from its rows 192..255, columns 0..127,
                // turned around in registers and put where CTA 0 would have put it (the slot layout does not change).  Both CTAs
                // then drain 50 chunks instead of 58 and 42, and the drain -- bound by each SM's 30 B/clk store path while the
                // tensor pipe waits -- is as long as its longer half.
                const bool diag = (seg.I == seg.J);
                const int ra_begin = diag ? row0 : 0;
                const int ra_end = (diag && rank == 0) ? min(cols_valid, kDiagSplitCol) : cols_valid;
                const int rb_end = (diag && rank == 1 && row0 >= kDiagSplitCol) ? min(cols_valid, kBlock) : 0;   // columns [0, rb_end)
                const int n_chunks_a = max((ra_end - ra_begin + 31) / 32, 0);
                const int n_chunks_r = n_chunks_a + (rb_end + 31) / 32;
                const int n_chunks = n_chunks_r + (cols_valid + 31) / 32;       // R chunks, then Q chunks (32 columns each)
                auto chunk_col = [&](int ch) {
                    return (ch < n_chunks_a) ? (ra_begin + 32 * ch) : (ch < n_chunks_r) ? 32 * (ch - n_chunks_a) : (256 + 32 * (ch - n_chunks_r));
                };
                auto chunk_load = [&](int ch, uint32_t (&v)[32]) {
                    ptx::tmem_ld_32x32(tmem_base + ((quarter * 32u) << 16) + (uint32_t)chunk_col(ch), v);
                };
                int32_t *slot_peer_cols = p.acc + ((size_t)seg.slot * 2 + 0) * (size_t)kAccElemsPerCta + (size_t)(row0 >> 2) * (32 * 4);
                auto chunk_store = [&](int ch, uint32_t (&v)[32]) {
                    const bool turned = ch >= n_chunks_a && ch < n_chunks_r;      // CTA 1's share of G[0:128, 128:256], see above
                    const uint32_t m = lane & 3u, quad = lane & ~3u;
                    if (turned) {
                        // turned around in registers: the four lanes of a quad (rows j = 4 g .. 4 g + 3 of this warp) exchange
                        // 4 x 4 blocks, after which lane (g, m) holds in v[4 t .. 4 t + 3], for row i = 4 t + m of the chunk, the
                        // four columns 4 g .. 4 g + 3 -- 16 bytes of CTA 0's slot each, 64 contiguous bytes per quad.  Register
                        // indices stay static: a lane rotates its block row by m before sending, the received column by -m after.
                        auto rot4 = [&](uint32_t (&a)[4], uint32_t by) {         // a[c] <- a[(c + by) & 3]
                            if (by & 1u) { const uint32_t t0 = a[0]; a[0] = a[1]; a[1] = a[2]; a[2] = a[3]; a[3] = t0; }
                            if (by & 2u) { const uint32_t t0 = a[0], t1 = a[1]; a[0] = a[2]; a[1] = a[3]; a[2] = t0; a[3] = t1; }
                        };
#pragma unroll
                        for (int t = 0; t < 8; ++t) {
                            uint32_t u[4] = {v[4 * t], v[4 * t + 1], v[4 * t + 2], v[4 * t + 3]};
                            rot4(u, m);                                           // u[r] = this row's column 4 t + ((m + r) & 3)
                            uint32_t o[4];
                            o[0] = u[0];                                          // own row, column 4 t + m
#pragma unroll
                            for (int r = 1; r < 4; ++r)                           // from lane (m - r) & 3: its row, column 4 t + m
                                o[r] = __shfl_sync(0xFFFFFFFFu, u[r], (int)(quad + ((m - (uint32_t)r) & 3u)));
                            uint32_t w[4] = {o[0], o[3], o[2], o[1]};             // o[r] is source row (m - r) & 3;  w[c] = row (m + c) & 3
                            rot4(w, (4u - m) & 3u);                               // w[c] <- row c
                            v[4 * t] = w[0]; v[4 * t + 1] = w[1]; v[4 * t + 2] = w[2]; v[4 * t + 3] = w[3];
                        }
                    }
                    // where vector g (v[4 g .. 4 g + 3]) of this lane goes inside the 4 KiB chunk [col / 4][row][col % 4]:
                    // as loaded, lane = row and g = column group; turned, (lane / 4) = column group and 4 g + m = row
                    const uint32_t vec0 = turned ? (lane >> 2) * 512u + m * 16u : lane * 16u;      // bytes
                    const uint32_t vec_step = turned ? 64u : 512u;
                    int32_t *chunk = turned ? slot_peer_cols + (size_t)(chunk_col(ch) >> 5) * (size_t)kAccElemsPerQuarter
                                            : slot_warp + (size_t)(chunk_col(ch) >> 2) * (32 * 4);
                    if (p.first_frame) {
                        // first frame of an integration: plain stores straight from the registers -- 16 bytes per lane and
                        // instruction, 512 (turned: 8 x 64) contiguous bytes of the slot per warp; no staging, no proxy fence, no
                        // bulk group
                        int32_t *dst = chunk + (vec0 >> 2);
#pragma unroll
                        for (int g = 0; g < 8; ++g)
                            ptx::st_global_v4(dst + g * (int)(vec_step >> 2), (int32_t)v[4 * g], (int32_t)v[4 * g + 1], (int32_t)v[4 * g + 2], (int32_t)v[4 * g + 3]);
                        return;
                    }
                    // later frames: the chunk is staged in shared memory in its final order and handed to ONE bulk int32 reduce-add
                    // (the addition happens at the destination, nothing is loaded into the SM).  Two staging buffers per warp;
                    // lane 0 owns the bulk groups.
                    const uint32_t stage = smem_epistage + (quarter * 2u + (uint32_t)(epi_chunks & 1u)) * Cfg::kEpiStageBytes;
                    if (lane == 0) ptx::bulk_wait_read<1>();       // the copy that last read this buffer (two chunks ago) is done with it
                    __syncwarp();
#pragma unroll
                    for (int g = 0; g < 8; ++g)
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(stage + vec0 + (uint32_t)g * vec_step), "r"(v[4 * g]),
                                     "r"(v[4 * g + 1]), "r"(v[4 * g + 2]), "r"(v[4 * g + 3])
                                     : "memory");
                    ptx::fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        ptx::bulk_reduce_add_s32(chunk, stage, Cfg::kEpiStageBytes);
                        ptx::bulk_commit();
                    }
                    ++epi_chunks;
                };
                // two register buffers: the TMEM load of chunk k+1 is in flight while chunk k is written out
                uint32_t va[32], vb[32];
                if (n_chunks > 0) chunk_load(0, va);
                for (int ch = 0; ch < n_chunks; ch += 2) {
                    ptx::tmem_wait_ld();
                    if (ch + 1 < n_chunks) chunk_load(ch + 1, vb); else release_tmem();
                    chunk_store(ch, va);
                    if (ch + 1 < n_chunks) {
                        ptx::tmem_wait_ld();
                        if (ch + 2 < n_chunks) chunk_load(ch + 2, va); else release_tmem();
                        chunk_store(ch + 1, vb);
                    }
                }
            }
            if (!released) release_tmem();
        }
        if (lane == 0) ptx::bulk_wait_all();                     // the slot is complete in global memory before the grid ends
    }

    // ---- teardown: everyone in both CTAs done with TMEM / peer smem before dealloc and exit ----
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::cluster_sync();
    if (warp == kWarpTmem) {
        ptx::tc_fence_after_sync();
        ptx::tmem_dealloc<2>(tmem_base, kAccCols);
    }
}

}  // namespace xc
