// Host planner: decode contexts -> page-granular KV splits, chunk -> query tiles
// (x KV splits when there are too few tiles to fill the GPU), one work list for the persistent kernel.
// Pure integer host code: depends only on lengths (never on page ids), so the GPU result is bit-identical
// under page permutation.
#include <algorithm>
#include <cstdint>

#include "kairos_internal.h"

namespace kairos {

namespace {
constexpr int kMinSplitPages = 4;      // never cut a KV range into pieces shorter than this
// Item costs in units of a quarter decode page (~550 SM cycles), from the CTA timelines under profiles/: a gen-1 chunk
// tile-page (N = 64 softmax on the critical path) costs ~1.5 decode pages, and every item carries a fixed cost
// (Q load, pipeline fill, epilogue: ~3k cycles for a decode split, ~9k for a chunk tile).  Only the ORDER of the queue
// (longest first) and the chunk / decode interleave depend on the fixed parts.
constexpr int kChunkCostNum = 6;
constexpr int kChunkCostDen = 4;
constexpr int kDecItemFixedCost = 5;
constexpr int kChunkItemFixedCost = 16;

inline int32_t ceil_div(int64_t a, int64_t b) { return int32_t((a + b - 1) / b); }

// Cost model of the SM sharing between the pair kernel (chunk) and the decode grid, in nominal SM cycles (1.965 GHz),
// calibrated on B200 (profiles/r01_bench_gen3.md): one 8-token tile x 64-key page on a pair (at the clocks the chip
// sustains under tensor load), the fixed cost of a tile (Q load, pipeline fill, epilogue), one decode page on one CTA
// when HBM is not the limit, the HBM floor per decode page with every SM streaming, and the same 8-token tile-page done
// as two gen-1 tiles (what the pair path has to beat).
constexpr int64_t kPairPageCycles = 1800;
constexpr int64_t kPairItemCycles = 27000;
constexpr int64_t kDecPageCycles = 2600;
constexpr int64_t kDecPageHbmSmCycles = 4260;
constexpr int32_t kGen1MaxTiles = 16;
constexpr int64_t kGen1MaxDecPages = 512;  // ... and only beside little decode work (long decodes want every SM streaming early)
constexpr int64_t kKernelFloorCycles = 25000;  // launch, first loads, first chain, epilogue of a persistent kernel (~12.7 us)

// When the chunk runs on the pair kernel, clusters are launched for EVERY SM pair (up to one per tile) and the two grids
// share the SMs in time: the decode grid is launched first on `dec_ctas` SMs (as 2-CTA clusters, so that it occupies whole
// TPCs), the clusters that do not fit beside it become resident when the decode CTAs exit and join the tile queue
// then.  dec_ctas = 0 means the decode grid is launched behind the pair grid with one CTA per SM and fills the SMs the
// clusters leave as they finish (the chunk is so much larger than the decode work that a static share would idle).
void choose_pairs(const int32_t* dec_ctx_lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len, int32_t ctas,
                  int32_t pair_mode, int32_t T2, Plan* plan) {
    if (pair_mode == 0 || chunk_len <= 0 || ctas < 2) return;
    const int32_t n_tiles = ceil_div(chunk_len, T2);
    int64_t pair_pages = 0;
    for (int32_t t = 0; t < n_tiles; ++t)
        pair_pages += ceil_div(int64_t(prefix_len) + std::min(chunk_len, (t + 1) * T2), kPage);
    int64_t dec_pages = 0;
    for (int32_t i = 0; i < n_dec; ++i) dec_pages += ceil_div(dec_ctx_lens[i], kPage);
    const int32_t max_pairs = std::min(n_tiles, ctas / 2);
    if (max_pairs < 1) return;
    // A chunk of at most kGen1MaxTiles 8-token tiles keeps too few SM pairs busy: it rides in the decode queue as 4-token
    // gen-1 tiles (KV-split across CTAs).  Anything larger runs on clusters: measured over a (B, K, C, P) grid off the five
    // BASELINE configs (profiles/r02_planner_offpoints.md), gen-1 tiles lose up to 1.9x there and win only below ~128 tokens.
    if (pair_mode == -1 && n_tiles <= kGen1MaxTiles && dec_pages <= kGen1MaxDecPages) return;
    const int64_t work_c = pair_pages * kPairPageCycles + int64_t(n_tiles) * kPairItemCycles;
    int32_t dec_ctas = 0;
    int32_t n_p = max_pairs;
    if (pair_mode < -1) {
        // forced (sweeps): -(n + 1) = n clusters first, the decode grid on every SM behind them
        n_p = std::min(-pair_mode - 1, max_pairs);
    } else if (n_dec > 0) {
        const int64_t td_all = dec_pages * kDecPageHbmSmCycles / ctas;  // decode alone, every SM streaming
        // (A) decode first on ctas - 2c SMs, c clusters beside it, every cluster afterwards
        auto t_dec_first = [&](int32_t c) {
            const int64_t td = std::max(dec_pages * kDecPageCycles / (ctas - 2 * c), td_all);
            return td + std::max<int64_t>(0, work_c - int64_t(c) * td) / max_pairs;
        };
        // (B) n clusters first, the decode grid (one CTA per SM) behind them: it takes the other SMs at once and the
        // clusters' SMs as they finish; n = max_pairs means the decode CTAs only fill the clusters' tail
        auto t_pairs_first = [&](int32_t n) {
            const int64_t tiles_each = ceil_div(n_tiles, n);
            const int64_t tc = std::max(work_c / n, tiles_each * (work_c / n_tiles));
            const int64_t done = std::min<int64_t>({dec_pages, tc * (ctas - 2 * n) / kDecPageCycles, tc * ctas / kDecPageHbmSmCycles});
            return tc + (dec_pages - done) * kDecPageHbmSmCycles / ctas;
        };
        int64_t best = -1;
        int32_t best_c = 0, best_n = 0;  // exactly one of them ends up > 0
        if (pair_mode > 0) {
            best_c = std::min({pair_mode, max_pairs, (ctas - 2) / 2});
            if (pair_mode >= max_pairs) { best_c = 0; best_n = max_pairs; }
        } else if (ceil_div(work_c, (td_all + kKernelFloorCycles) * 4 / 10) <= std::min(max_pairs, 48)) {
            // a chunk that is small beside the decode work (measured: configs[3] C <= 1024): just enough clusters to finish
            // it within ~40 % of the decodes' time, launched first (fewer clusters gain 1-3 % when the estimate is right and
            // lose > 10 % when it is not, profiles/r02_planner_offpoints.md); the decode grid (the
            // decode-only instantiation with the deeper ring) streams on the other SMs and inherits theirs
            best_n = std::max(std::min(8, max_pairs), ceil_div(work_c, (td_all + kKernelFloorCycles) * 4 / 10));
        } else {
            // decode first only pays when the tiles outnumber the SM pairs at least twice (measured: with fewer tiles the
            // clusters that start late run alone at the end)
            // t_dec_first is flat in c once the decode CTAs stream below the HBM floor (td * (ctas - 2c) is constant), so the
            // tie decides: the LARGEST share of clusters whose decode grid still ends within 40 % of the estimate (the decode
            // CTAs stream at their best rate on few SMs, but short requests and a loaded L2 make them slower than
            // kDecPageCycles, and a decode grid that outlasts the chunk is the worst order of all).  Measured on a 90-point
            // (B, K, C, P) grid (profiles/r02_order_sweep.md): the planner's loss against the best forced order went from a
            // mean of 2.5 % (worst 19-26 %, three points above 10 %) to 1.8 % (worst 8 %).
            for (int32_t c = 1; n_tiles >= ctas && c <= std::min(max_pairs, (ctas - 2) / 2); ++c) {
                const int64_t td = std::max(dec_pages * kDecPageCycles / (ctas - 2 * c), td_all);
                const int64_t t = t_dec_first(c);
                const bool better = best < 0 || t * 1000 < best * 999;
                const bool tie = !better && t * 1000 <= best * 1001 && td * 5 <= t * 2;
                if (better || tie) { best = best < 0 ? t : std::min(best, t); best_c = c; best_n = 0; }
            }
            for (int32_t n = 1; n <= max_pairs; ++n) {
                const int64_t t = t_pairs_first(n);
                if (best < 0 || t < best) { best = t; best_c = 0; best_n = n; }
            }
            // a chunk that dwarfs the decode work: a static share idles (tile quantisation, contention) more than the overlap
            // gains; measured on configs[2] and [4] (profiles/r01_bench_gen3.md): the decode CTAs fill the clusters' tail instead
            if (work_c / max_pairs >= 4 * td_all) { best_c = 0; best_n = max_pairs; }
        }
        if (best_c > 0) dec_ctas = ctas - 2 * best_c;
        else n_p = best_n;
    } else if (pair_mode < 0) {
        // chunk only: one cluster per tile, up to one per SM pair
    } else {
        n_p = std::min(pair_mode, max_pairs);
    }
    plan->dec_ctas = dec_ctas;
    plan->n_pairs = n_p;
    for (int32_t t = 0; t < n_tiles; ++t) {
        WorkItem w{};
        w.kind = 1;
        w.q_index = t * T2;
        w.n_q = std::min(chunk_len, (t + 1) * T2) - t * T2;
        w.page_begin = 0;
        w.page_end = ceil_div(int64_t(prefix_len) + w.q_index + w.n_q, kPage);
        w.n_keys = prefix_len + w.q_index + 1;
        w.partial_slot = -1;
        w.cost = w.page_end;
        plan->pair_items.push_back(w);
    }
    std::stable_sort(plan->pair_items.begin(), plan->pair_items.end(), [](const WorkItem& a, const WorkItem& b) { return a.cost > b.cost; });
}
}  // namespace

void build_plan(const int32_t* dec_ctx_lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len,
                int32_t target_ctas, int32_t T, Plan* plan, int32_t pair_mode, int32_t T2) {
    plan->items.clear();
    plan->combines.clear();
    plan->pair_items.clear();
    plan->n_pairs = 0;
    plan->dec_ctas = 0;
    plan->n_decode_items = plan->n_chunk_items = plan->n_partial_slots = 0;
    if (target_ctas < 1) target_ctas = 1;
    choose_pairs(dec_ctx_lens, n_dec, chunk_len, prefix_len, target_ctas, pair_mode, T2, plan);
    if (plan->n_pairs > 0) {  // the chunk runs on SM pairs: the queue below holds decode splits only
        chunk_len = 0;
        if (plan->dec_ctas > 0) target_ctas = plan->dec_ctas;
    }

    // ---- total cost, in units of 4*decode-page
    int64_t dec_pages = 0;
    for (int32_t i = 0; i < n_dec; ++i) dec_pages += ceil_div(dec_ctx_lens[i], kPage);
    const int32_t n_tiles = chunk_len > 0 ? ceil_div(chunk_len, T) : 0;
    int64_t tile_pages = 0;
    for (int32_t t = 0; t < n_tiles; ++t) {
        int32_t q_last = std::min(chunk_len, (t + 1) * T) - 1;
        tile_pages += ceil_div(int64_t(prefix_len) + q_last + 1, kPage);
    }
    const int64_t total_cost = dec_pages * kChunkCostDen + tile_pages * kChunkCostNum;
    // An item should not exceed about half of one CTA's fair share -- 0.6 of it in a queue of decode splits alone, where
    // every split that is avoided saves a partial (32 KB written, read again by the combine): measured on configs[3] C = 0,
    // 256 x 32 pages on 148 CTAs, whole requests beside 24-page bodies run 113.9 -> 109.4 us against two halves each.
    const bool dec_queue_only = chunk_len == 0 && plan->n_pairs == 0;
    int64_t max_item_cost = dec_queue_only ? total_cost * 3 / (5 * int64_t(target_ctas)) : total_cost / (2 * int64_t(target_ctas));
    max_item_cost = std::max<int64_t>(max_item_cost, int64_t(kMinSplitPages) * kChunkCostDen);

    // global caps that keep the workspace bound of kairos_workspace_bytes valid
    int32_t dec_split_budget = 4 * target_ctas;   // extra decode partial slots beyond one per request
    int32_t chunk_slot_budget = 8 * target_ctas;  // chunk partial token-slots

    std::vector<WorkItem> dec_items, chunk_items;

    // ---- decode splits.  Two item sizes: "big" pieces (about half of one CTA's fair share) carry most of the
    // pages with few partials; a tail budget of kMinSplitPages-sized pieces, peeled off the longest requests, goes
    // to the END of the queue so that the dynamic queue's finishing imbalance is a few pages, not one big piece.
    {
        const int64_t fair_pages = std::max<int64_t>(1, total_cost / (int64_t(kChunkCostDen) * target_ctas));
        const int32_t big = int32_t(std::max<int64_t>(kMinSplitPages, std::min<int64_t>(max_item_cost / kChunkCostDen, dec_queue_only ? (fair_pages * 3 + 4) / 5 : (fair_pages + 1) / 2)));
        int64_t tail_budget = fair_pages >= 4 * kMinSplitPages ? int64_t(target_ctas) * 2 * kMinSplitPages : 0;  // pages
        std::vector<int32_t> order(n_dec);
        for (int32_t i = 0; i < n_dec; ++i) order[i] = i;
        std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return dec_ctx_lens[a] > dec_ctx_lens[b]; });
        std::vector<int32_t> cuts;
        for (int32_t oi = 0; oi < n_dec; ++oi) {
            const int32_t i = order[oi];
            const int32_t pages = ceil_div(dec_ctx_lens[i], kPage);
            // small tail pieces of this request (peeled from its end)
            int32_t n_small = 0;
            if (tail_budget > 0 && pages >= 3 * kMinSplitPages) {
                n_small = int32_t(std::min<int64_t>({int64_t(2), tail_budget / kMinSplitPages, int64_t(pages / kMinSplitPages - 2)}));
                n_small = std::max(n_small, 0);
            }
            const int32_t body = pages - n_small * kMinSplitPages;
            int32_t n_big = ceil_div(body, big);
            n_big = std::min(n_big, std::max(1, body / kMinSplitPages));
            int32_t n_splits = n_big + n_small;
            if (n_splits > 1 && n_splits - 1 > dec_split_budget) {  // workspace bound: fall back to fewer pieces
                n_small = 0;
                n_big = std::min(ceil_div(pages, big), 1 + std::max(0, dec_split_budget));
                n_big = std::max(1, std::min(n_big, std::max(1, pages / kMinSplitPages)));
                n_splits = n_big;
            }
            const int32_t body2 = pages - n_small * kMinSplitPages;
            cuts.clear();
            cuts.push_back(0);
            const int32_t per = ceil_div(body2, n_big);
            for (int32_t s = 1; s <= n_big; ++s) {
                const int32_t e = std::min(body2, s * per);
                if (e > cuts.back()) cuts.push_back(e);
            }
            for (int32_t s = 1; s <= n_small; ++s) cuts.push_back(body2 + s * kMinSplitPages);
            n_splits = int32_t(cuts.size()) - 1;
            if (n_splits > 1) dec_split_budget -= (n_splits - 1);
            tail_budget -= int64_t(n_small) * kMinSplitPages;
            int32_t first_slot = -1;
            if (n_splits > 1) {
                first_slot = plan->n_partial_slots;
                plan->n_partial_slots += n_splits;
                plan->combines.push_back(CombineItem{i, first_slot, n_splits, 0 /*decode*/ | (1 << 8) /*slot stride 1*/});
            }
            for (int32_t s = 0; s < n_splits; ++s) {
                WorkItem w{};
                w.kind = 0;
                w.q_index = i;
                w.page_begin = cuts[s];
                w.page_end = cuts[s + 1];
                w.n_keys = dec_ctx_lens[i];
                w.n_q = 1;
                w.partial_slot = n_splits > 1 ? first_slot + s : -1;
                w.cost = (w.page_end - w.page_begin) * kChunkCostDen + kDecItemFixedCost;
                dec_items.push_back(w);
            }
        }
    }

    // ---- chunk tiles (KV-split only while there are fewer tiles than CTAs)
    for (int32_t t = 0; t < n_tiles; ++t) {
        const int32_t q0 = t * T;
        const int32_t nq = std::min(chunk_len, q0 + T) - q0;
        const int32_t pages = ceil_div(int64_t(prefix_len) + q0 + nq, kPage);
        int32_t n_splits = 1;
        if (n_tiles < target_ctas) {
            int32_t max_pages = int32_t(std::max<int64_t>(kMinSplitPages, max_item_cost / kChunkCostNum));
            n_splits = ceil_div(pages, max_pages);
            n_splits = std::min(n_splits, std::max(1, pages / kMinSplitPages));
            if (n_splits > 1 && n_splits * T > chunk_slot_budget) n_splits = std::max(1, chunk_slot_budget / T);
            if (n_splits > 1) chunk_slot_budget -= n_splits * T;
        }
        const int32_t per = ceil_div(pages, n_splits);
        n_splits = ceil_div(pages, per);
        int32_t first_slot = -1;
        if (n_splits > 1) {
            first_slot = plan->n_partial_slots;
            plan->n_partial_slots += n_splits * T;  // layout [split][token]
            for (int32_t j = 0; j < nq; ++j)
                plan->combines.push_back(CombineItem{q0 + j, first_slot + j, n_splits, 1 /*chunk*/ | (T << 8)});
        }
        for (int32_t s = 0; s < n_splits; ++s) {
            WorkItem w{};
            w.kind = 1;
            w.q_index = q0;
            w.page_begin = s * per;
            w.page_end = std::min(pages, (s + 1) * per);
            w.n_keys = prefix_len + q0 + 1;
            w.n_q = nq;
            w.partial_slot = n_splits > 1 ? first_slot + s * T : -1;
            w.cost = (w.page_end - w.page_begin) * kChunkCostNum + kChunkItemFixedCost;
            chunk_items.push_back(w);
        }
    }

    auto by_cost = [](const WorkItem& a, const WorkItem& b) {
        if (a.cost != b.cost) return a.cost > b.cost;
        if (a.q_index != b.q_index) return a.q_index < b.q_index;
        return a.page_begin < b.page_begin;
    };
    std::sort(dec_items.begin(), dec_items.end(), by_cost);
    std::sort(chunk_items.begin(), chunk_items.end(), by_cost);

    // ---- interleave the two kinds in proportion to their total cost, so that at any time part of the
    // SMs stream decode pages from HBM while the others run chunk tiles on the tensor cores (a10).
    int64_t dc = 0, cc = 0, dtot = 0, ctot = 0;
    for (auto& w : dec_items) dtot += w.cost;
    for (auto& w : chunk_items) ctot += w.cost;
    size_t di = 0, ci = 0;
    plan->items.reserve(dec_items.size() + chunk_items.size());
    while (di < dec_items.size() || ci < chunk_items.size()) {
        bool take_chunk;
        if (di >= dec_items.size()) take_chunk = true;
        else if (ci >= chunk_items.size()) take_chunk = false;
        else take_chunk = (cc * dtot <= dc * ctot);  // cc/ctot <= dc/dtot: the chunk list is behind
        if (take_chunk) { cc += chunk_items[ci].cost; plan->items.push_back(chunk_items[ci++]); }
        else { dc += dec_items[di].cost; plan->items.push_back(dec_items[di++]); }
    }
    plan->n_decode_items = int32_t(dec_items.size());
    plan->n_chunk_items = int32_t(chunk_items.size());
}

}  // namespace kairos
