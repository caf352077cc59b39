// impl 1, chunk tiles of 8 query tokens (gen 2): a 2-CTA cluster splits the tile's two GEMMs over two SMs, because one
// SM's tensor memory cannot hold both accumulators of a 128-row MLA tile (O[128 x 512] fp32 is
// all 512 TMEM columns) and the swapped-operand single-CTA form is shared-memory-operand bound at <= 48 % of the
// tensor peak (profiles/r01_mma_issue_probe.txt).
//
//   rank 0, "S-CTA":  S[128 q rows x 64 keys] = Q[128 x 576] . K_page^T     tcgen05.mma M=128 N=64, A = Q held in TMEM
//                     (bf16, 288 columns, loaded once per tile through TMA staging), B = the K page in SMEM (K-major,
//                     TMA, 2 stages refilled in 3 groups); 4 softmax warps own one query row per thread (row max / sum
//                     are thread-local); P = exp2(S*c - m) as bf16 and the per-row rescale factors are staged in local
//                     shared memory and moved to the O-CTA by cp.async.bulk (shared::cta -> shared::cluster), which
//                     completes on the O-CTA's mbarrier.
//   rank 1, "O-CTA":  O[128 x 512] += P[128 x 64] . V_page[64 x 512]        tcgen05.mma M=128 N=256 x2, A = P (SMEM,
//                     K-major), B = the latent page as stored (MN-major, TMA, 3 stages), fp32 accumulators = all
//                     512 TMEM columns; its 4 row-owning warps rescale O on the (rare, thresholded) running-max updates
//                     and write O / l as bf16.
//
// Rows of a tile: r = 16 * (token in tile) + head.  Work items come from a queue shared by all pairs (rank 0 pops and
// forwards the index through DSMEM).  Same definition as the gen-1 path; parity-tested against the oracle.
#include <cuda_bf16.h>

#include <algorithm>

#include "kairos_internal.h"
#include "umma_ptx.cuh"

namespace kairos {
namespace {
using namespace ptx;

constexpr int kPairTileTokens = 8;
constexpr int kPairThreads = 192;            // warp 0 TMA producer (+ queue on rank 0), warp 1 MMA issuer, warps 2-5 softmax / epilogue
constexpr int kKStage = kPage * kTokenBytes;  // 73,728: K page, all 576 dims (S-CTA)
constexpr int kVStage = kPage * kLatent * 2;  // 65,536: latent part only (O-CTA)
constexpr int kStages = 3;                    // V stages of the O-CTA
constexpr int kStagesK = 2;                   // K stages of the S-CTA (the rest of its shared memory stages P for the bulk copy)
constexpr int kOffPStage = kStagesK * kKStage; // S-CTA: local P staging, 2 x 16 KB
constexpr int kPBytes = 128 * 128;            // P[128 rows][64 keys] bf16, SWIZZLE_128B K-major
constexpr int kOffP = kStages * kVStage;      // O-CTA: P buffers after the V stages
constexpr int kOffQStage = kStagesK * kKStage + 2 * kPBytes + 2048;  // S-CTA: two 16 KB TMA landing buffers for Q chunks (1024-aligned)
static_assert(kOffQStage % 1024 == 0, "SWIZZLE_128B tiles need 1024-byte alignment");
constexpr int kOffSmallS = kOffQStage + 2 * 16384;  // P staging + alpha staging (1 KB) + linv staging (512 B)
constexpr int kOffSmallO = kStages * kVStage + 2 * kPBytes;  // 229,376
constexpr int kPairSmallBytes = 2048;
constexpr int kPairSmem = (kOffSmallO > kOffSmallS ? kOffSmallO : kOffSmallS) + kPairSmallBytes + 1024;
static_assert(kPairSmem <= 232448, "exceeds the per-CTA shared memory limit");

constexpr uint32_t kColQ = 0;     // S-CTA TMEM: Q as the A operand, 288 columns (2 bf16 per column)
constexpr uint32_t kColS2 = 320;  // S-CTA TMEM: S accumulators at 320 and 384 (64 columns each)
constexpr float kRescaleThreshold2 = 8.0f;
constexpr float kLn2b = 0.6931471805599453f;
constexpr float kMinusHuge2 = -1.0e30f;

// S-CTA only (lives in its otherwise unused shared memory at kOffSmallS): one barrier pair per slot of the K ring (a group
// of chunks of one page); a slot is refilled as soon as its MMAs retire.
constexpr int kGroupChunks = 3;  // chunks per ring slot (24 KB): an mbarrier wait costs the issuing warp ~100 cycles even when
                                 // complete, so per-chunk slots (9 waits per page) made the MMA warp issue-bound
constexpr int kGroups = 9 / kGroupChunks;
struct ScRing {
    uint64_t kv_full[kStagesK * kGroups], kv_empty[kStagesK * kGroups];
};
static_assert(kOffSmallS + int(sizeof(ScRing)) <= kOffSmallO, "ScRing overlaps the shared small struct");

// One struct for both ranks (same offsets in both CTAs, so mapa of a local address names the peer's copy).
struct PairSmall {
    // S-CTA
    uint64_t s_full[2], s_empty[2], q_ready, q_free;
    uint64_t p_empty[2];   // arrived by the O-CTA's tcgen05.commit when PV(g) has consumed P buffer g & 1
    uint64_t fin_empty;    // arrived by the O-CTA's epilogue warps: linv[] may be overwritten
    uint64_t item_empty[2];
    uint64_t qst_full[4];  // Q chunk landed in a landing buffer (TMA)
    // O-CTA
    uint64_t v_full[kStages], v_empty[kStages], p_full[2], corr_done[2], pv_done[2], o_full, o_empty, fin_full;
    // both
    uint64_t item_full[2];
    int32_t item_ring[2];
    uint32_t tmem_base;
    alignas(16) float alpha[2][128];  // O-CTA: per-row O rescale factors of page g (bulk-copied with P; 1 = none)
    alignas(16) float linv[128];      // O-CTA: 1 / l per row at the end of the item (bulk-copied)
};
static_assert(sizeof(PairSmall) <= kPairSmallBytes, "PairSmall does not fit");


struct PairParams {
    const WorkItem* items;
    int32_t n_items;
    int32_t* counter;      // queue head of the pair kernel
    int32_t* done_counter; // finished clusters (last one re-arms the queue)
    const int32_t* chunk_pt;
    const __nv_bfloat16* q_chunk;
    __nv_bfloat16* out_chunk;
    float* lse_chunk;
    float scale_log2;
};

__device__ __forceinline__ WorkItem load_item2(const WorkItem* p) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(p));
    const int4 b = __ldg(reinterpret_cast<const int4*>(p) + 1);
    WorkItem w;
    w.kind = a.x; w.q_index = a.y; w.page_begin = a.z; w.page_end = a.w;
    w.n_keys = b.x; w.n_q = b.y; w.partial_slot = b.z; w.cost = b.w;
    return w;
}
__device__ __forceinline__ void tma_load_box3(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int32_t row, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5}], [%2], %6;"
        ::"r"(smem_u32(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(0), "r"(row), "r"(0),
          "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tma_load_chunk(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int32_t row, int32_t chunk,
                                               uint64_t policy) {  // box (64 elems, 64 rows, kGroupChunks chunks)
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5}], [%2], %6;"
        ::"r"(smem_u32(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(0), "r"(row), "r"(chunk),
          "l"(policy)
        : "memory");
}
__device__ __forceinline__ float ex2f(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t pack2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
// ------------------------------------------------------------------------------------------------------------
// S-CTA, softmax warps (128 threads, thread = query row `row` = TMEM lane).  peer_* are shared::cluster addresses in
// the O-CTA.  g counts pages over the whole kernel (S buffer / P buffer = g & 1), `it` counts items.
// ------------------------------------------------------------------------------------------------------------
// S-CTA: Q tile of item `it` -> TMEM (the 128 row-owning threads).  Waits for the S-MMAs of item it - 1 (q_free).
// The tile [128 rows x 576] moves through FOUR 16 KB landing buffers, one TMA box (64 dims x 128 rows, SWIZZLE_128B, rows past
// the chunk's end zero-filled) per 64-dim chunk: the two dedicated Q buffers and the two P staging buffers, which are idle
// between the last P of one item and the first P of the next.  `g` = global page counter of the item's first page: P
// buffer g & 1 last carried page g - 2 and buffer (g + 1) & 1 page g - 1; each may be overwritten once the O-CTA's PV of
// that page has retired (p_empty: by then the bulk copy that read the buffer has completed as well).  With 3-4 boxes in
// flight the load is ~3k cycles instead of ~7k with two (it is the serial part of every tile boundary).
__device__ __forceinline__ void sc_load_q(PairSmall* sm, uint8_t* pstage, const WorkItem& w, const PairParams& p, const CUtensorMap* qmap,
                                          uint32_t tmem, int row, int q4, int lane, uint32_t& qcount, uint32_t it, uint32_t g) {
    const uint32_t lane_base = uint32_t(q4 * 32) << 16;
    uint8_t* qst = reinterpret_cast<uint8_t*>(sm) - kOffSmallO + kOffQStage;
    uint8_t* buf[4] = {qst, qst + 16384, pstage + (g & 1u) * kPBytes, pstage + ((g + 1u) & 1u) * kPBytes};
    const int row0 = w.q_index * kHeads;
    auto issue = [&](int c) {  // row 0 only
        const int bi = c & 3;
        if (c == 2) mbar_wait(&sm->p_empty[g & 1u], ((g >> 1) & 1u) ^ 1u);
        if (c == 3) mbar_wait(&sm->p_empty[(g + 1u) & 1u], (((g + 1u) >> 1) & 1u) ^ 1u);
        if (c == 2 || c == 3) fence_proxy_async_smem();  // the buffer's last writes came from this CTA's threads (generic proxy)
        mbar_arrive_expect_tx(&sm->qst_full[bi], 16384);
        tma_load_2d(buf[bi], qmap, &sm->qst_full[bi], c * 64, row0, kEvictFirst);
    };
    if (row == 0) {  // the first boxes start moving before the previous item's S-MMAs have retired
        issue(0);
        issue(1);
        issue(2);
    }
    mbar_wait(&sm->q_free, (it & 1) ^ 1);  // previous item's S-MMAs have retired
    tc_fence_after();
#pragma unroll 1
    for (int c = 0; c < 9; ++c) {
        const uint32_t bi = c & 3;
        mbar_wait(&sm->qst_full[bi], (qcount >> bi) & 1);  // qcount: one phase-parity bit per landing buffer
        qcount ^= 1u << bi;
        // each thread reads its own row's 128 B (conflict free) and stores 32 TMEM columns
        const uint8_t* src = buf[bi] + row * 128;
        uint32_t r[32];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const uint4 v = *reinterpret_cast<const uint4*>(src + ((j ^ (row & 7)) << 4));
            r[4 * j + 0] = v.x; r[4 * j + 1] = v.y; r[4 * j + 2] = v.z; r[4 * j + 3] = v.w;
        }
        tmem_st32(tmem + lane_base + kColQ + 32 * c, r);
        if (c == 0 || c + 4 < 9) {
            asm volatile("bar.sync 3, 128;" ::: "memory");  // every row has read this buffer
            if (row == 0) {
                if (c == 0) issue(3);  // the fourth buffer frees last (PV of the previous item's last page)
                if (c + 4 < 9) issue(c + 4);
            }
        }
    }
    tmem_wait_st();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->q_ready);
}

__device__ __forceinline__ WorkItem sc_fetch_item(PairSmall* sm, const PairParams& p, int lane, uint32_t it, int* idx_out) {
    const uint32_t slot = it & 1, iph = (it >> 1) & 1;
    mbar_wait(&sm->item_full[slot], iph);
    const int idx = *reinterpret_cast<volatile int32_t*>(&sm->item_ring[slot]);
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->item_empty[slot]);
    *idx_out = idx;
    WorkItem w{};
    if (idx >= 0) w = load_item2(p.items + idx);
    return w;
}

// Processes item `it` (its Q is already in TMEM), then fetches item it + 1 and loads that item's Q.
__device__ __forceinline__ void sc_softmax_item(PairSmall* sm, uint8_t* pstage, uint32_t peer_small, uint32_t peer_p, const WorkItem& w,
                                                const PairParams& p, const CUtensorMap* qmap, uint32_t tmem, int row, int q4, int lane,
                                                uint32_t& g, uint32_t& qcount, uint32_t it, WorkItem* next, int* next_idx) {
    const int tok = row >> 4, head = row & 15;
    const uint32_t lane_base = uint32_t(q4 * 32) << 16;
    float m_ref = kMinusHuge2, l = 0.f;
    const int npages = w.page_end - w.page_begin;
    const int vis = w.n_keys + tok;  // keys visible to this row: positions < vis
    for (int pg = 0; pg < npages; ++pg, ++g) {
        const uint32_t b = g & 1, ph = (g >> 1) & 1;
        mbar_wait(&sm->s_full[b], ph);
        tc_fence_after();
        float x[64];
        tmem_ld32(tmem + lane_base + kColS2 + b * 64, reinterpret_cast<uint32_t*>(x));
        tmem_ld32(tmem + lane_base + kColS2 + b * 64 + 32, reinterpret_cast<uint32_t*>(x) + 32);
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->s_empty[b]);

        const int key0 = (w.page_begin + pg) * kPage;
        const bool boundary = key0 + kPage > w.n_keys;  // some row of the tile does not see every key of this page
        float tm = -INFINITY;
        if (boundary) {
#pragma unroll
            for (int k = 0; k < 64; ++k) {
                x[k] = (key0 + k < vis) ? x[k] * p.scale_log2 : -INFINITY;
                tm = fmaxf(tm, x[k]);
            }
        } else {
#pragma unroll
            for (int k = 0; k < 64; ++k) {
                x[k] *= p.scale_log2;
                tm = fmaxf(tm, x[k]);
            }
        }
        // thresholded running max: the reference moves only when the page's max exceeds it by more than 2^8
        const bool need = tm - m_ref > kRescaleThreshold2;
        float alpha = 1.f;
        if (need) {
            alpha = ex2f(m_ref - tm);  // 0 on the first visible page (m_ref = -1e30)
            l *= alpha;
            m_ref = tm;
        }
        float sum = 0.f;
#pragma unroll
        for (int k = 0; k < 64; ++k) {
            x[k] = ex2f(x[k] - m_ref);
            sum += x[k];
        }
        l += sum;
        // ---- P row (bf16, 128 B) -> O-CTA shared memory, K-major SWIZZLE_128B: row r at r*128, 16-B chunk c at c ^ (r & 7)
        // p_empty is a remote tcgen05.commit: it orders nothing but the re-use of this CTA's own staging buffer, whose reader
        // (this CTA's bulk copy) finished before the PV that is being signalled started.  A CTA-scope wait is enough; the
        // acquire.cluster form makes ptxas emit CCTL.IVALL (an L1 invalidate, long-scoreboard) after EVERY poll -- ncu: 5 % of
        // all samples here and 30 % at the O-CTA's p_full wait below.
        mbar_wait(&sm->p_empty[b], ph ^ 1);
        // local staging (K-major SWIZZLE_128B: row r at r*128, 16-B chunk c at c ^ (r & 7)), then one 4 KB bulk copy per
        // warp into the O-CTA's P buffer, completing on its p_full mbarrier (DSMEM moves ~20 B/clk: asynchronous, so the
        // softmax threads do not wait for it)
        uint8_t* prow = pstage + b * kPBytes + row * 128;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            uint4 v;
            v.x = pack2(x[8 * c + 0], x[8 * c + 1]);
            v.y = pack2(x[8 * c + 2], x[8 * c + 3]);
            v.z = pack2(x[8 * c + 4], x[8 * c + 5]);
            v.w = pack2(x[8 * c + 6], x[8 * c + 7]);
            *reinterpret_cast<uint4*>(prow + ((c ^ (row & 7)) << 4)) = v;
        }
        // rescale factor of this row for the O-CTA (1 = leave O alone; on the first page O is overwritten, accumulate = 0):
        // staged next to P and bulk-copied too, so the per-page path has no generic-proxy remote store at all
        reinterpret_cast<float*>(pstage + 2 * kPBytes)[b * 128 + row] = pg > 0 ? alpha : 1.f;
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
            const uint32_t bar = peer_small + uint32_t(offsetof(PairSmall, p_full)) + b * 8;
            asm volatile("mbarrier.arrive.expect_tx.relaxed.cluster.shared::cluster.b64 _, [%0], %1;" ::"r"(bar), "r"(4096u + 128u) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(peer_p + b * kPBytes + uint32_t(q4) * 4096u), "r"(smem_u32(pstage + b * kPBytes + q4 * 4096)), "r"(4096u), "r"(bar)
                         : "memory");
            asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(peer_small + uint32_t(offsetof(PairSmall, alpha)) + (b * 128 + q4 * 32) * 4),
                           "r"(smem_u32(pstage + 2 * kPBytes + (b * 128 + q4 * 32) * 4)), "r"(128u), "r"(bar)
                         : "memory");
        }
    }
    // ---- end of item: 1 / l to the O-CTA's epilogue; lse from here
    mbar_wait_cluster(&sm->fin_empty, (it & 1) ^ 1);
    {  // staged locally and bulk-copied like P (a release.cluster arrive per thread costs ~3000 cycles)
        float* lst = reinterpret_cast<float*>(pstage + 2 * kPBytes + 1024);
        lst[row] = 1.f / l;
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
            const uint32_t bar = peer_small + uint32_t(offsetof(PairSmall, fin_full));
            asm volatile("mbarrier.arrive.expect_tx.relaxed.cluster.shared::cluster.b64 _, [%0], %1;" ::"r"(bar), "r"(128u) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(peer_small + uint32_t(offsetof(PairSmall, linv)) + q4 * 128), "r"(smem_u32(lst + q4 * 32)), "r"(128u), "r"(bar)
                         : "memory");
        }
    }
    if (tok < w.n_q && p.lse_chunk) p.lse_chunk[size_t(w.q_index + tok) * kHeads + head] = (m_ref + log2f(l)) * kLn2b;
    // Every S-MMA of this item has retired (its last s_full was consumed above): Q may be replaced.  The next item's Q is
    // loaded only now, after the last P and 1/l have left, so that the ~7k-cycle load overlaps the O-CTA's last PV and its
    // epilogue (which otherwise stall the next item's first pages) instead of delaying them.
    *next = sc_fetch_item(sm, p, lane, it + 1, next_idx);
    if (*next_idx >= 0) sc_load_q(sm, pstage, *next, p, qmap, tmem, row, q4, lane, qcount, it + 1, g);
}

// S-CTA, MMA warp (converged; one elected lane issues)
__device__ __forceinline__ void sc_mma_item(PairSmall* sm, ScRing* ring, uint32_t tmem, uint32_t kv_base, int npages, uint32_t& g, uint32_t it,
                                            const PairParams& p) {
    constexpr uint32_t idesc = make_idesc_bf16(128, 64, 0, 0);
    constexpr uint32_t hi = smem_desc_hi(1024);
    mbar_wait(&sm->q_ready, it & 1);
    tc_fence_after();
    for (int pg = 0; pg < npages; ++pg, ++g) {
        const uint32_t st = g % kStagesK, sph = (g / kStagesK) & 1, b = g & 1, bph = (g >> 1) & 1;
        mbar_wait(&sm->s_empty[b], bph ^ 1);
        const uint32_t kb_lo = smem_desc_lo(kv_base + st * kKStage, 16);
        mbar_wait(&ring->kv_full[st * kGroups], sph);
        tc_fence_after();
#pragma unroll
        for (uint32_t gr = 0; gr < kGroups; ++gr) {
#pragma unroll
            for (uint32_t cc = 0; cc < kGroupChunks; ++cc) {
                const uint32_t c = gr * kGroupChunks + cc;
#pragma unroll
                for (uint32_t j = 0; j < 4; ++j)
                    umma_bf16_ts_lohi(tmem + kColS2 + b * 64, tmem + kColQ + (c * 4 + j) * 8, kb_lo + ((c * 8192 + j * 32) >> 4), hi,
                                      idesc, (c | j) != 0);
            }
            umma_commit_elect(&ring->kv_empty[st * kGroups + gr]);
        }
        umma_commit_elect(&sm->s_full[b]);
    }
    umma_commit_elect(&sm->q_free);
}

// ------------------------------------------------------------------------------------------------------------
// O-CTA, correction + epilogue warps (128 threads, thread = query row = TMEM lane)
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void oc_epilogue_item(PairSmall* sm, uint8_t* v_stages, uint32_t peer_small, const WorkItem& w, const PairParams& p,
                                                 uint32_t tmem, int row, int q4, int lane, uint32_t& g, uint32_t it) {
    const uint32_t lane_base = uint32_t(q4 * 32) << 16;
    const int npages = w.page_end - w.page_begin;
    for (int pg = 0; pg < npages; ++pg, ++g) {
        const uint32_t b = g & 1, ph = (g >> 1) & 1;
        {
            // Keys that no row of the tile sees (stale slots of the sequence's last page) have P = 0, but the PV MMA still
            // multiplies their V rows, and 0 * NaN = NaN: zero those rows of the landed V stage (128 B per 64-dim chunk; the
            // 128-byte swizzle permutes inside a row).  Thread = (token row & 63, half of the 8 chunks).
            const int key0 = (w.page_begin + pg) * kPage, vis_max = w.n_keys + w.n_q - 1;
            if (key0 + kPage > vis_max) {
                const uint32_t st = g % kStages;
                mbar_wait(&sm->v_full[st], (g / kStages) & 1);
                const int t = row & 63;
                if (key0 + t >= vis_max) {
                    uint8_t* vst = v_stages + st * kVStage + t * 128;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        uint4* dst = reinterpret_cast<uint4*>(vst + ((row >> 6) * 4 + c) * 8192);
#pragma unroll
                        for (int j = 0; j < 8; ++j) dst[j] = make_uint4(0u, 0u, 0u, 0u);
                    }
                }
                fence_proxy_async_smem();
            }
        }
        mbar_wait(&sm->p_full[b], ph);  // P and alpha arrive through the async proxy (complete_tx): the TMA pattern, CTA-scope wait
        const float a = *reinterpret_cast<volatile float*>(&sm->alpha[b][row]);
        if (__any_sync(0xffffffffu, a != 1.f)) {  // warp-uniform: tcgen05.ld / st are warp-collective
            // a row's reference max moved: every PV issued so far must have landed before O is rescaled
            mbar_wait(&sm->pv_done[(g - 1) & 1], ((g - 1) >> 1) & 1);
            tc_fence_after();
#pragma unroll 1
            for (int c = 0; c < 16; ++c) {
                uint32_t r[32];
                tmem_ld32(tmem + lane_base + c * 32, r);
                tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 32; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * a);
                tmem_st32(tmem + lane_base + c * 32, r);
            }
            tmem_wait_st();
            tc_fence_before();
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->corr_done[b]);
    }
    // ---- epilogue: O / l -> bf16
    mbar_wait(&sm->o_full, it & 1);
    mbar_wait(&sm->fin_full, it & 1);  // 1 / l arrives through the async proxy as well
    tc_fence_after();
    const float linv = *reinterpret_cast<volatile float*>(&sm->linv[row]);
    {
        // Each thread owns one output row; writing 16 B per row per instruction would touch 32 cache lines per store
        // (measured: ~14k cycles per tile).  A 4x4 transpose of 16-B units inside every lane quad makes each store
        // instruction write 64 contiguous bytes per row, 8 rows per instruction.
        const int qd = lane & 3;
        const int rbase = row - qd;  // first row of this quad
        __nv_bfloat16* obase = p.out_chunk + (size_t(w.q_index) * kHeads) * kLatent;
        // the tcgen05.ld of block c + 1 is in flight while block c is converted, transposed and stored
        auto emit = [&](const uint32_t (&r)[32], int c) {
            uint4 e[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                e[j].x = pack2(__uint_as_float(r[8 * j + 0]) * linv, __uint_as_float(r[8 * j + 1]) * linv);
                e[j].y = pack2(__uint_as_float(r[8 * j + 2]) * linv, __uint_as_float(r[8 * j + 3]) * linv);
                e[j].z = pack2(__uint_as_float(r[8 * j + 4]) * linv, __uint_as_float(r[8 * j + 5]) * linv);
                e[j].w = pack2(__uint_as_float(r[8 * j + 6]) * linv, __uint_as_float(r[8 * j + 7]) * linv);
            }
#pragma unroll
            for (int m = 1; m <= 2; m <<= 1) {
                const bool up = (qd & m) != 0;
#pragma unroll
                for (int a = 0; a < 4; ++a) {
                    if (a & m) continue;
                    const uint4 snd = up ? e[a] : e[a ^ m];
                    uint4 rcv;
                    rcv.x = __shfl_xor_sync(0xffffffffu, snd.x, m);
                    rcv.y = __shfl_xor_sync(0xffffffffu, snd.y, m);
                    rcv.z = __shfl_xor_sync(0xffffffffu, snd.z, m);
                    rcv.w = __shfl_xor_sync(0xffffffffu, snd.w, m);
                    if (up) e[a] = rcv; else e[a ^ m] = rcv;
                }
            }
            // e[i] now holds 16-B unit `qd` of row rbase + i
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int rr = rbase + i;
                if ((rr >> 4) < w.n_q)
                    *reinterpret_cast<uint4*>(obase + size_t(rr) * kLatent + c * 32 + qd * 8) = e[i];
            }
        };
        uint32_t ra[32], rb[32];
        tmem_ld32(tmem + lane_base, ra);
#pragma unroll 1
        for (int c = 0; c < 16; c += 2) {
            tmem_wait_ld();
            tmem_ld32(tmem + lane_base + (c + 1) * 32, rb);
            emit(ra, c);
            tmem_wait_ld();
            if (c + 2 < 16) tmem_ld32(tmem + lane_base + (c + 2) * 32, ra);
            emit(rb, c + 1);
        }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) {
        mbar_arrive(&sm->o_empty);
        mbar_arrive_remote(peer_small + uint32_t(offsetof(PairSmall, fin_empty)));
    }
}

// O-CTA, MMA warp
__device__ __forceinline__ void oc_mma_item(PairSmall* sm, uint32_t peer_small, uint32_t tmem, uint32_t v_base, uint32_t p_base,
                                            int npages, uint32_t& g, uint32_t it, const PairParams& p) {
    constexpr uint32_t idesc = make_idesc_bf16(128, 256, 0, 1);  // A = P K-major, B = V page MN-major
    constexpr uint32_t hi = smem_desc_hi(1024);
    for (int pg = 0; pg < npages; ++pg, ++g) {
        const uint32_t st = g % kStages, sph = (g / kStages) & 1, b = g & 1, bph = (g >> 1) & 1;
        mbar_wait(&sm->corr_done[b], bph);
        mbar_wait(&sm->v_full[st], sph);
        if (pg == 0) mbar_wait(&sm->o_empty, (it & 1) ^ 1);  // previous item's epilogue has drained O
        fence_proxy_async_smem();  // P arrived through the generic proxy of the peer's threads
        tc_fence_after();
        const uint32_t pa_lo = smem_desc_lo(p_base + b * kPBytes, 16);
        const uint32_t vb_lo = smem_desc_lo(v_base + st * kVStage, 8192);
#pragma unroll
        for (uint32_t hf = 0; hf < 2; ++hf)
#pragma unroll
            for (uint32_t ks = 0; ks < 4; ++ks)
                umma_bf16_ss_lohi(tmem + hf * 256, pa_lo + ((ks * 32) >> 4), hi, vb_lo + ((hf * 4 * 8192 + ks * 2048) >> 4), hi, idesc,
                                  (pg > 0 || ks > 0));
        umma_commit_elect(&sm->v_empty[st]);
        umma_commit_elect(&sm->pv_done[b]);
        umma_commit_elect_addr(peer_small + uint32_t(offsetof(PairSmall, p_empty)) + b * 8);
        if (pg == npages - 1) umma_commit_elect(&sm->o_full);
    }
}

// ------------------------------------------------------------------------------------------------------------
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kPairThreads, 1)
kairos_chunk_pair_kernel(const __grid_constant__ CUtensorMap pool_map_k, const __grid_constant__ CUtensorMap pool_map_v,
                         const __grid_constant__ CUtensorMap q_map, const PairParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t rank = cluster_ctarank();  // 0 = S-CTA, 1 = O-CTA
    PairSmall* sm = reinterpret_cast<PairSmall*>(base + kOffSmallO);  // same offset on both ranks (beyond both layouts)
    ScRing* ring = reinterpret_cast<ScRing*>(base + kOffSmallS);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t peer_small = mapa_shared(smem_u32(sm), rank ^ 1);
    const uint32_t peer_p = mapa_shared(smem_u32(base + kOffP), 1);  // P buffers live in the O-CTA

    if (threadIdx.x == 0) {
        for (int i = 0; i < kStagesK * kGroups; ++i) {
            mbar_init(&ring->kv_full[i], 1);
            mbar_init(&ring->kv_empty[i], 1);
        }
        for (int i = 0; i < kStages; ++i) {
            mbar_init(&sm->v_full[i], 1);
            mbar_init(&sm->v_empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&sm->s_full[i], 1);
            mbar_init(&sm->s_empty[i], 4);
            mbar_init(&sm->p_empty[i], 1);
            mbar_init(&sm->p_full[i], 4);
            mbar_init(&sm->corr_done[i], 4);
            mbar_init(&sm->pv_done[i], 1);
            mbar_init(&sm->item_full[i], 1);
            mbar_init(&sm->item_empty[i], 11);  // S-CTA: MMA warp + 4 softmax warps; O-CTA: producer + MMA + 4 epilogue warps
        }
        for (int i = 0; i < 4; ++i) mbar_init(&sm->qst_full[i], 1);
        mbar_init(&sm->q_ready, 4);
        mbar_init(&sm->q_free, 1);
        mbar_init(&sm->fin_empty, 4);
        mbar_init(&sm->fin_full, 4);
        mbar_init(&sm->o_full, 1);
        mbar_init(&sm->o_empty, 4);
        fence_barrier_init();
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // a decode grid queued behind this kernel may take SMs as clusters finish
    if (warp == 0 && lane == 0) prefetch_tensormap(rank == 0 ? &pool_map_k : &pool_map_v);
    if (warp == 2 && lane == 0 && rank == 0) prefetch_tensormap(&q_map);
    if (warp == 1) tmem_alloc(&sm->tmem_base, 512);
    tc_fence_before();
    __syncthreads();
    cluster_arrive();  // the peer's barriers are initialised before anything arrives on them
    cluster_wait();
    tc_fence_after();
    const uint32_t tmem = sm->tmem_base;

    if (warp == 0) {
        // ================= producer: (rank 0) pops the queue and forwards the index; both ranks TMA-load their pages
        uint32_t g = 0;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1, iph = (it >> 1) & 1;
            int idx = 0;
            if (rank == 0) {
                if (lane == 0) {
                    // Every item comes from the queue, the first one too.  A static first item (cluster i takes item i, as in the
                    // decode grid) was measured and dropped: in the decode-first launch orders half of the clusters only become
                    // resident when decode CTAs exit, and the long tiles at the head of the list (longest first) would wait for
                    // them (configs[1] 48.7 -> 53 us, configs[3] C = 2048 175.6 -> 187 us).
                    idx = atomicAdd(p.counter, 1);
                    if (idx >= p.n_items) idx = -1;
                    mbar_wait_cluster(&sm->item_empty[slot], iph ^ 1);
                    sm->item_ring[slot] = idx;
                    st_cluster_b32(peer_small + uint32_t(offsetof(PairSmall, item_ring)) + slot * 4, uint32_t(idx));
                    mbar_arrive(&sm->item_full[slot]);
                    mbar_arrive_remote(peer_small + uint32_t(offsetof(PairSmall, item_full)) + slot * 8);
                }
                idx = __shfl_sync(0xffffffffu, idx, 0);
            } else {
                mbar_wait_cluster(&sm->item_full[slot], iph);
                idx = *reinterpret_cast<volatile int32_t*>(&sm->item_ring[slot]);
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(peer_small + uint32_t(offsetof(PairSmall, item_empty)) + slot * 8);
            }
            if (idx < 0) break;
            const WorkItem w = load_item2(p.items + idx);
            if (rank == 0 && lane == 0) {  // the tile's Q rows are contiguous: bring them into L2 one item ahead of their use
                const uint32_t qbytes = uint32_t(w.n_q) * kHeads * kTokenBytes;
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p.q_chunk + size_t(w.q_index) * kHeads * kDim), "r"(qbytes) : "memory");
            }
            const int32_t* pt = p.chunk_pt + w.page_begin;
            const int npages = w.page_end - w.page_begin;
            for (int i = 0; i < npages; i += 32) {
                const int my = (i + lane < npages) ? __ldg(pt + i + lane) : 0;
                const int cnt = min(32, npages - i);
                for (int j = 0; j < cnt; ++j, ++g) {
                    const int pid = __shfl_sync(0xffffffffu, my, j);
                    if (lane == 0) {
                        const uint32_t ns = rank == 0 ? kStagesK : kStages;
                        const uint32_t st = g % ns, sph = (g / ns) & 1;
                        if (rank == 0) {
                            // one full barrier per page (a completed mbarrier wait costs the MMA warp ~100 cycles), one empty
                            // barrier per group of chunks (a group is refilled as soon as its MMAs retire)
                            for (int gr = 0; gr < kGroups; ++gr) {
                                mbar_wait(&ring->kv_empty[st * kGroups + gr], sph ^ 1);
                                if (gr == 0) mbar_arrive_expect_tx(&ring->kv_full[st * kGroups], kKStage);
                                tma_load_chunk(base + st * kKStage + gr * kGroupChunks * 8192, &pool_map_k, &ring->kv_full[st * kGroups],
                                               pid * kPage, gr * kGroupChunks, kEvictLast);
                            }
                        } else {
                            mbar_wait(&sm->v_empty[st], sph ^ 1);
                            mbar_arrive_expect_tx(&sm->v_full[st], kVStage);
                            tma_load_box3(base + st * kVStage, &pool_map_v, &sm->v_full[st], pid * kPage, kEvictLast);
                        }
                    }
                }
            }
        }
    } else {
        // ================= consumers: MMA warp (1) and the four row-owning warps (2-5)
        const int q4 = warp & 3;  // TMEM lane quadrant this warp may touch
        const int row = q4 * 32 + lane;
        uint32_t g = 0, qcount = 0;
        if (rank == 0 && warp >= 2) {
            // S-CTA row-owning warps: item fetch and Q load run one item ahead of the softmax
            int idx;
            WorkItem w = sc_fetch_item(sm, p, lane, 0, &idx);
            if (idx >= 0) sc_load_q(sm, base + kOffPStage, w, p, &q_map, tmem, row, q4, lane, qcount, 0, 0);
            for (uint32_t it = 0; idx >= 0; ++it) {
                WorkItem nxt{};
                int nidx = -1;
                sc_softmax_item(sm, base + kOffPStage, peer_small, peer_p, w, p, &q_map, tmem, row, q4, lane, g, qcount, it, &nxt, &nidx);
                w = nxt;
                idx = nidx;
            }
        } else {
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it & 1, iph = (it >> 1) & 1;
                int idx;
                if (rank == 0) {
                    mbar_wait(&sm->item_full[slot], iph);
                    idx = *reinterpret_cast<volatile int32_t*>(&sm->item_ring[slot]);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&sm->item_empty[slot]);
                } else {
                    mbar_wait_cluster(&sm->item_full[slot], iph);
                    idx = *reinterpret_cast<volatile int32_t*>(&sm->item_ring[slot]);
                    __syncwarp();
                    if (lane == 0) mbar_arrive_remote(peer_small + uint32_t(offsetof(PairSmall, item_empty)) + slot * 8);
                }
                if (idx < 0) break;
                const WorkItem w = load_item2(p.items + idx);
                const int npages = w.page_end - w.page_begin;
                if (warp == 1) {
                    if (rank == 0) sc_mma_item(sm, ring, tmem, smem_u32(base), npages, g, it, p);
                    else oc_mma_item(sm, peer_small, tmem, smem_u32(base), smem_u32(base + kOffP), npages, g, it, p);
                } else {
                    oc_epilogue_item(sm, base, peer_small, w, p, tmem, row, q4, lane, g, it);
                }
            }
        }
    }

    // ---- teardown: neither CTA may exit while its peer can still touch its shared memory
    tc_fence_before();
    __syncthreads();
    // launched behind the decode grid with programmatic stream serialisation: wait for that grid before exiting, so that this
    // grid's completion implies the decode grid's for everything that follows in the stream (no-op for an ordinary launch)
    if (threadIdx.x == 0) asm volatile("griddepcontrol.wait;" ::: "memory");
    cluster_arrive();
    cluster_wait();
    if (warp == 1) tmem_dealloc(tmem, 512);
    if (threadIdx.x == 0 && rank == 0) {
        __threadfence();
        const int prev = atomicAdd(p.done_counter, 1);
        if (prev == int(gridDim.x / 2) - 1) {  // last pair out re-arms the queue for the next launch (stream-ordered)
            *p.counter = 0;
            *p.done_counter = 0;
        }
    }
}

}  // namespace

int pair_tile_tokens() { return kPairTileTokens; }

int pair_init(kairos_ctx* ctx) {
    typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                      const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                      CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    KAIROS_CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    if (!fn || q != cudaDriverEntryPointSuccess) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    // latent part of a page: pool viewed as [chunk 9][row num_pages*64][64 elems], box = 8 chunks x 64 rows x 64 elems
    cuuint64_t dims[3] = {64, cuuint64_t(ctx->cfg.num_pages) * kPage, 9};
    cuuint64_t strides[2] = {cuuint64_t(kTokenBytes), 128};
    cuuint32_t box[3] = {64, 64, 8};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(&ctx->pool_map_v, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, ctx->cfg.pool, dims, strides,
                                                     box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled(pool, latent box) failed: " + std::to_string(int(r)));
    cuuint32_t box1[3] = {64, 64, kGroupChunks};  // a group of 64-dim chunks of a page: the S-CTA's K ring is refilled group by group
    r = reinterpret_cast<EncodeTiledFn>(fn)(&ctx->pool_map_c, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, ctx->cfg.pool, dims, strides, box1, es,
                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled(pool, chunk box) failed: " + std::to_string(int(r)));
    KAIROS_CUDA_TRY(cudaFuncSetAttribute(kairos_chunk_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairSmem));
    return KAIROS_OK;
}

// Launches n_pairs 2-CTA clusters over the chunk-tile items (kind 1, 8-token tiles, no KV split) on `stream`.
int launch_attn_pair(kairos_ctx* ctx, const StepArgs& a, const WorkItem* dev_items, int32_t n_items, int32_t n_pairs,
                     cudaStream_t stream, bool pdl) {
    PairParams p;
    p.items = dev_items;
    p.n_items = n_items;
    p.counter = reinterpret_cast<int32_t*>(ctx->cfg.workspace) + 2;
    p.done_counter = reinterpret_cast<int32_t*>(ctx->cfg.workspace) + 3;
    p.chunk_pt = a.chunk_page_table;
    p.q_chunk = reinterpret_cast<const __nv_bfloat16*>(a.q_chunk);
    p.out_chunk = reinterpret_cast<__nv_bfloat16*>(a.out_chunk);
    p.lse_chunk = a.lse_chunk;
    p.scale_log2 = ctx->cfg.softmax_scale * 1.4426950408889634f;
    n_pairs = std::max(1, std::min(n_pairs, n_items));
    const CUtensorMap& q_map = ctx->qp_map.map;  // q_chunk as [C*16 rows][576], box = 64 dims x 128 rows (encoded by the caller)
    // pdl: launched right behind the decode grid on the same stream with programmatic stream serialisation, so that the
    // clusters start as soon as every decode CTA is resident (that kernel triggers launch_dependents at its start) and
    // run beside it; neither kernel reads what the other writes, so this kernel only executes griddepcontrol.wait before it exits.
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(2 * n_pairs), 1, 1);
    cfg.blockDim = dim3(kPairThreads, 1, 1);
    cfg.dynamicSmemBytes = kPairSmem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kairos_chunk_pair_kernel, ctx->pool_map_c, ctx->pool_map_v, q_map, p));
    return KAIROS_OK;
}

}  // namespace kairos
