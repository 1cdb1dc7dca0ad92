// schedule.hpp -- host-side work decomposition for the persistent X-engine kernel (pure C++, no CUDA).
//
// Work item  = one super-tile (f, I <= J) over the whole frame; it is cut along time into STAGES of
//              kStageT samples.  Cost model per stage: 16 for an off-diagonal item (2 x 4 MMAs of 128 clk: the kernel runs at
//              the tensor pipe's floor) and 9 for a diagonal one (2 x 2 MMAs would be 8; in the N > 256
//              kernel, whose rings are sized for the off-diagonal form, the diagonal stages run a little above their
//              floor).  Measured, not only counted -- xcorr_process (us) at C4 / C5 by diagonal cost: 8: 558 / 1266,
//              9: 547 / 1201, 10: 551 / 1218, 11 (the model of the earlier, issue-bound kernel): 561 / 1280.  N <= 256 has
//              diagonal items only, any constant does.  (A per-segment cost for the accumulator drain, during which the
//              worker's tensor pipe idles, was tried on top: no measurable gain at C2..C5, left out.)
// Worker     = one CTA pair (two SMs, one 2-CTA tcgen05 MMA stream); there are `n_workers` of them.
//
// Hybrid data-parallel / stream-K split (integer addition is exact and order independent, so a
// super-tile may be summed by several workers, each adding its partial into the accumulator):
//   * whole rounds of n_workers items go round-robin, whole, to the workers, as long as that leaves no worker
//     above the mean load of the whole job -- consecutive items (same channel, neighbouring super-tiles) run at
//     the same time on different workers, so blocks shared between them are served by L2;
//   * the stages of the remaining items are dealt out as contiguous runs so that every worker ends
//     with (nearly) the same total cost ("water filling").
// Every (item, stage) is assigned to exactly one worker (checked by tests/test_host_logic.py).
// Each segment owns one accumulator SLOT (layout.hpp); a tile's slots are numbered contiguously.
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>

namespace xc {

constexpr int kStageT = 64;  // time samples per pipeline stage (MMA K-steps of 32)

struct Segment {          // 32 bytes, read by the kernel
    int32_t f;            // channel
    int32_t I, J;         // super-block row / column (I <= J)
    int32_t stage_begin;  // [stage_begin, stage_end) in units of kStageT samples
    int32_t stage_end;
    int32_t tile;         // f * n_supertiles + supertile_index(I, J)
    int32_t slot;         // accumulator slot owned by this segment (layout.hpp)
    int32_t pad1;
};

struct Schedule {
    int n_workers = 0;
    int n_stages = 0;                 // stages per item = ceil(T / kStageT)
    std::vector<Segment> segments;    // grouped by worker
    std::vector<int32_t> worker_begin;  // size n_workers + 1, offsets into segments
    std::vector<int32_t> tile_slot_begin;  // size n_tiles + 1: slots [b[t], b[t+1]) belong to tile t
};

inline Schedule make_schedule(int n_inputs, int n_freq, int n_time, int n_workers)
{
    Schedule s;
    s.n_workers = n_workers;
    s.n_stages = (n_time + kStageT - 1) / kStageT;
    const int nb = (n_inputs + 255) / 256;
    const int nst = nb * (nb + 1) / 2;

    struct Item { int f, I, J, tile; int64_t cost_per_stage; };   // cost model: see the header
    std::vector<Item> items;
    items.reserve((size_t)n_freq * nst);
    for (int f = 0; f < n_freq; ++f)
        for (int I = 0; I < nb; ++I)
            for (int J = I; J < nb; ++J)
                items.push_back({f, I, J, f * nst + (I * (2 * nb - I + 1) / 2 + (J - I)), I == J ? 9 : 16});

    const int64_t n_items = (int64_t)items.size();
    // whole rounds of n_workers items go data-parallel only as long as no worker ends above the mean load of the whole job
    // (2 % slack): an item dearer than the mean (N = 512, T long: one off-diagonal item per worker is 8192 of a mean of 7085)
    // has to be cut, so there the water filling takes everything
    int64_t total_cost = 0;
    for (const Item &it : items) total_cost += it.cost_per_stage * s.n_stages;
    const int64_t cap = total_cost / n_workers + total_cost / n_workers / 50 + 4;
    int64_t n_dp = 0;
    {
        std::vector<int64_t> trial(n_workers, 0);
        for (int64_t r = 0; (r + 1) * n_workers <= n_items; ++r) {
            int64_t mx = 0;
            for (int w = 0; w < n_workers; ++w) {
                trial[w] += items[r * n_workers + w].cost_per_stage * s.n_stages;
                mx = std::max(mx, trial[w]);
            }
            if (mx > cap) break;
            n_dp = (r + 1) * n_workers;
        }
    }
    std::vector<std::vector<Segment>> per(n_workers);
    std::vector<std::vector<Segment>> per_dp(n_workers);   // the whole items of the data-parallel rounds
    std::vector<int64_t> load(n_workers, 0);

    for (int64_t u = 0; u < n_dp; ++u) {
        const Item &it = items[u];
        const int w = (int)(u % n_workers);
        per_dp[w].push_back({it.f, it.I, it.J, 0, s.n_stages, it.tile, 0, 0});
        load[w] += it.cost_per_stage * s.n_stages;
    }

    // remainder: water-fill
    int64_t rem_cost = 0;
    for (int64_t u = n_dp; u < n_items; ++u) rem_cost += items[u].cost_per_stage * s.n_stages;
    if (rem_cost > 0) {
        // level L with sum_w max(0, L - load[w]) == rem_cost  (bisection on integers, then exact shares)
        int64_t lo = *std::min_element(load.begin(), load.end());
        int64_t hi = *std::max_element(load.begin(), load.end()) + rem_cost;
        while (lo < hi) {
            const int64_t mid = lo + (hi - lo) / 2;
            int64_t cap = 0;
            for (int w = 0; w < n_workers; ++w) cap += std::max<int64_t>(0, mid - load[w]);
            if (cap >= rem_cost) hi = mid; else lo = mid + 1;
        }
        std::vector<int64_t> share(n_workers);
        int64_t total = 0;
        for (int w = 0; w < n_workers; ++w) { share[w] = std::max<int64_t>(0, lo - load[w]); total += share[w]; }
        // trim the surplus (total >= rem_cost) from the last workers with a share
        for (int w = n_workers - 1; w >= 0 && total > rem_cost; --w) {
            const int64_t cut = std::min(share[w], total - rem_cost);
            share[w] -= cut; total -= cut;
        }
        // walk the remaining stages in order, handing out contiguous runs
        int w = 0;
        int64_t boundary = share[0];  // cumulative cost position where worker w's run ends
        int64_t pos = 0;
        for (int64_t u = n_dp; u < n_items; ++u) {
            const Item &it = items[u];
            int st = 0;
            while (st < s.n_stages) {
                while (w < n_workers - 1 && pos >= boundary) { ++w; boundary += share[w]; }
                // stages of this item that start before `boundary`
                int64_t room = boundary - pos;
                int take = (w == n_workers - 1) ? (s.n_stages - st)
                                                : (int)std::min<int64_t>(s.n_stages - st, (room + it.cost_per_stage - 1) / it.cost_per_stage);
                if (take <= 0) take = 1;
                per[w].push_back({it.f, it.I, it.J, st, st + take, it.tile, 0, 0});
                load[w] += it.cost_per_stage * take;
                pos += it.cost_per_stage * take;
                st += take;
            }
        }
    }

    // Order inside a worker.  N > 256: the data-parallel rounds first -- all workers start them together, so neighbouring
    // super-tiles of a channel walk through time side by side and share their blocks through L2.  N <= 256 (nothing to
    // share): the worker's FIRST water-filled piece, then its whole items, then the rest -- that piece is the tail of an
    // item and its length differs from worker to worker (the cut points of the water filling fall anywhere), so all later
    // item boundaries, where an SM drains its accumulators at 30 B/clk, are spread over the item period instead of hitting
    // L2 from all 148 SMs at once.
    for (int w = 0; w < n_workers; ++w) {
        const size_t at = (nb > 1 || per[w].empty()) ? 0 : 1;
        per[w].insert(per[w].begin() + at, per_dp[w].begin(), per_dp[w].end());
    }

    // slots: one per segment, numbered in (tile, stage_begin) order so that a tile's slots are contiguous
    {
        std::vector<Segment *> all;
        for (auto &v : per) for (auto &g : v) all.push_back(&g);
        std::sort(all.begin(), all.end(), [](const Segment *a, const Segment *b) {
            return a->tile != b->tile ? a->tile < b->tile : a->stage_begin < b->stage_begin;
        });
        const int n_tiles = n_freq * nst;
        s.tile_slot_begin.assign(n_tiles + 1, 0);
        for (size_t k = 0; k < all.size(); ++k) { all[k]->slot = (int32_t)k; s.tile_slot_begin[all[k]->tile + 1] += 1; }
        for (int t = 0; t < n_tiles; ++t) s.tile_slot_begin[t + 1] += s.tile_slot_begin[t];
    }

    s.worker_begin.resize(n_workers + 1);
    for (int w = 0; w < n_workers; ++w) {
        s.worker_begin[w] = (int32_t)s.segments.size();
        s.segments.insert(s.segments.end(), per[w].begin(), per[w].end());
    }
    s.worker_begin[n_workers] = (int32_t)s.segments.size();
    return s;
}

}  // namespace xc
