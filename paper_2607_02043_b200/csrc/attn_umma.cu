// impl 1 (the product path): persistent, warp-specialised tcgen05 / TMA / TMEM kernel for the mixed step.
//
// One CTA per SM pops work items (decode KV splits and prefill-chunk tiles) from one
// queue.  Both item kinds run the same "swapped operand" pipeline on one 64-token page per iteration, because all
// 16 heads of a token share one latent tile (BASELINE.json north_star):
//
//   S^T[64 keys x N]  = K_page[64 x 576] . Q^T[576 x N]      tcgen05.mma M=64,  K-major A (page) and B (queries)
//   P^T = exp2(S^T*c - m)  (column statistics across the 64 key lanes, lazy max update)
//   O^T[512 x N]     += V^T[512 x 64] . P^T[64 x N]          tcgen05.mma M=128 x4, MN-major A = the SAME smem page
//
//   N = 16 query rows (1 decode token x 16 heads) or 64 (4 chunk tokens x 16 heads).  A page is loaded once by five TMA
//   boxes (4 pairs of latent chunks + the RoPE chunk, SWIZZLE_128B, 8 KB slots of [64 tokens][128 B]) into a ring of
//   slots and serves as K (K-major) and as V (MN-major).  Accumulators live in TMEM: S^T double-buffered (2 x 64 columns),
//   O^T 4 x 64 columns, fp32.
//
// Warp roles (320 threads): warp 0 = TMA producer + work-queue pop, warp 1 = MMA issuer (one elected lane) + TMEM owner,
// warps 2-9 = softmax / correction / epilogue (two per TMEM lane quadrant, half of the query columns each).
// Two instantiations: <false> holds a 64-row chunk Q tile and 18 slots, <true> (queues without chunk tiles) two 16-row decode
// Q buffers and 22 slots.  Descriptor encodings were validated on B200 by profiles/r01_tcgen05_probe.txt; DESIGN.md 6.1 has
// the measurements behind the structure.
#include <cuda_bf16.h>

#include <algorithm>
#include <cstdlib>

#include "kairos_internal.h"
#include "umma_ptx.cuh"

namespace kairos {
namespace {
using namespace ptx;

constexpr int kSoftmaxWarps = 8;                 // 2 per TMEM lane quadrant: each takes half of the query-row columns
constexpr int kSoftmaxThreads = kSoftmaxWarps * 32;
constexpr int kThreads = 64 + kSoftmaxThreads + 32;  // warp 0 producer, warp 1 S issuer, warps 2-9 softmax, warp 10 PV issuer
constexpr int kPvWarp = 2 + kSoftmaxWarps;
constexpr int kChunkTileTokens = 4;
// one page = 73,728 B = 9 slots of 8 KB ([64 tokens][128 B], SWIZZLE_128B)
constexpr int kSlotBytes = 8192;
// Shared memory: the Q tile, then a ring of 8 KB slots that pages stream through (9 consecutive slots per page, refilled
// as pages retire, so that more than two pages' worth of loads can be in flight), then the barriers / statistics.
// DEC = true is the decode-only instantiation: two 16-row Q buffers (36 KB) leave room for 22 slots (2.44 pages in flight);
// the mixed instantiation holds a 64-row Q tile (72 KB) and 18 slots.  Decode items alternate between two 18 KB Q
// buffers at the start of the Q region (item parity), so that the next item's Q is loaded while the current item still
// streams its pages; a chunk tile takes the whole region (both buffers).
constexpr int kDecPBytes = 2048;
template <bool DEC>
struct Geo {
    static constexpr int kQBytes = (DEC ? 2 * 16 : 64) * kTokenBytes;  // two decode Q buffers, or one 64-row chunk tile
    static constexpr int kSlots = DEC ? 22 : 18;  // even: a pair of latent slots (one M=128 V^T operand) never straddles the wrap
    static constexpr int kOffKV = kQBytes;
    static constexpr int kOffP = kOffKV + kSlots * kSlotBytes;  // DEC: two 2 KB P buffers ([16 query rows][64 keys], K-major)
    static constexpr int kOffSmall = kOffP + (DEC ? 2 * kDecPBytes : 0);
    static constexpr int kSmemBytes = kOffSmall + 3072 + 1024;  // Small + alignment slack
    static_assert(kQBytes % 1024 == 0 && kSlots % 2 == 0, "ring must stay 1024-B aligned and even");
    static_assert(kSmemBytes <= 232448, "exceeds the per-CTA shared memory limit");
};
constexpr int kOffQ = 0;
constexpr int kDecQBytes = 16 * kTokenBytes;  // 18,432: one decode Q buffer
constexpr int kSmallBytes = 3072;
constexpr int kPageRing = 4;  // full / empty barriers per page in flight (at most 4 pages have slots in the ring at once)

// Where page number g (counted per CTA since launch) sits in a ring of R slots: it takes slots s .. s+8 (mod R), s = 9g mod R.
// The 8 latent slots start at the even one of {s, s+1} so that slot pairs (one 128-dim V^T block) are contiguous; the RoPE
// slot is the remaining one (before the latent slots when s is odd, after them when s is even).  P^T [64 keys][<=64 rows]
// bf16 (8 KB) is written into the page's RoPE slot: that slot is only read by the S MMAs, which have completed before the
// softmax of the page starts, and the page's slots are not reloaded until the PV MMAs that read P^T have completed.
struct PageSlots {
    uint32_t pair[4];  // first slot of latent chunks (2b, 2b+1)
    uint32_t rope;
    uint32_t odd;      // s is odd: the RoPE slot comes first in ring order
};
template <int R>
__device__ __forceinline__ PageSlots page_slots(uint32_t g) {
    PageSlots ps;
    const uint32_t s = (g * 9u) % uint32_t(R);
    ps.odd = s & 1u;
    const uint32_t e = s + ps.odd;
    ps.rope = ps.odd ? s : (s + 8u) % uint32_t(R);
#pragma unroll
    for (uint32_t b = 0; b < 4; ++b) ps.pair[b] = (e + 2u * b) % uint32_t(R);
    return ps;
}

constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0;    // S^T buffers at columns 0 and 64
constexpr uint32_t kColO = 128;  // O^T blocks at 128 + 64*b
constexpr float kRescaleThreshold = 8.0f;  // log2 units: rescale O only when the max grows by more than 2^8
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kMinusHuge = -1.0e30f;  // finite stand-in for "no key seen yet" (keeps x - m free of inf - inf)

struct Small {
    uint64_t q_full[2], q_empty[2], kv_full[kPageRing][5], kv_empty[kPageRing][5], s_full[2], s_empty[2], p_full[2], pv_done[2], o_full, o_empty;
    uint64_t item_full[2], item_empty[2];
    int32_t item_ring[2];
    uint32_t tmem_base;
    uint32_t pad;
    float m_ref[64];   // running reference max per query row (log2 domain); -1e30 while nothing visible yet
    float alpha[64];   // O / l rescale factor decided for the current page
    float red[4][64];  // per-warp column maxima (per page) / column sums (epilogue)
    float linv[64];
};
static_assert(sizeof(Small) <= kSmallBytes, "Small does not fit");


struct KParams {
    const WorkItem* items;
    int32_t n_items;
    int32_t* counters;  // [0] queue head, [1] finished CTAs
    const int32_t* dec_pt;
    int32_t dec_stride;
    const int32_t* chunk_pt;
    __nv_bfloat16* out_dec;
    __nv_bfloat16* out_chunk;
    float* lse_dec;
    float* lse_chunk;
    uint8_t* partials;
    float scale_log2;
    int32_t static_first;  // 1: CTA b starts with item b and the queue hands out items from gridDim.x on
};

__device__ __forceinline__ WorkItem load_item(const WorkItem* p) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(p));
    const int4 b = __ldg(reinterpret_cast<const int4*>(p) + 1);
    WorkItem w;
    w.kind = a.x; w.q_index = a.y; w.page_begin = a.z; w.page_end = a.w;
    w.n_keys = b.x; w.n_q = b.y; w.partial_slot = b.z; w.cost = b.w;
    return w;
}

__device__ __forceinline__ void tma_load_chunks(uint32_t smem_dst, const CUtensorMap* map, uint64_t* bar, int32_t row, int32_t chunk,
                                                uint64_t policy) {
    // 3-D box (64 elems, 64 rows, 1 or 2 chunks) of the pool viewed as [chunk][row][64]: lands as [chunks][64][128 B]
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5}], [%2], %6;"
        ::"r"(smem_dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(0), "r"(row), "r"(chunk),
          "l"(policy)
        : "memory");
}

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float warp_max(float v) {
    float r;
    asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
}
__device__ __forceinline__ void named_sync(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(kSoftmaxThreads) : "memory"); }
__device__ __forceinline__ bool named_or(int id, bool pred) {
    uint32_t r;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t"
        "setp.ne.u32 p, %1, 0;\n\t"
        "bar.red.or.pred q, %2, %3, p;\n\t"
        "selp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(r)
        : "r"(uint32_t(pred)), "r"(id), "n"(kSoftmaxThreads)
        : "memory");
    return r != 0;
}
// partial (split) results are re-read by the combine kernel right after this kernel: keep them in L2
__device__ __forceinline__ void st_f32_evict_last(float* p, float v) {
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(kEvictLast) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// ------------------------------------------------------------------------------------------------------------
// softmax / correction / epilogue for one work item; N = 16 (decode) or 64 (chunk tile) query rows.
// 8 warps: warp sw works on TMEM lane quadrant sw & 3 (16 of its lanes hold the M=64 accumulator rows = keys) and on
// the column half sw >> 2 (N/2 query rows).
// ------------------------------------------------------------------------------------------------------------
template <int N, int R, bool PK>
__device__ __forceinline__ void softmax_item(Small* sm, uint8_t* kv, const WorkItem& w, const KParams& p, uint32_t tmem,
                                             int sw, int lane, uint32_t& g, uint32_t it) {
    constexpr int NC = N / 2;            // columns of this warp
    constexpr int W = NC < 16 ? NC : 16;  // columns per tcgen05.ld
    const int w4 = (sw + 2) & 3;         // TMEM lane quadrant of CTA warp 2 + sw (a warp may only touch lanes 32*(warp%4)..)
    const int cbase = (sw >> 2) * NC;
    const int tid_s = sw * 32 + lane;
    const bool lane_ok = lane < 16;       // M=64 accumulator rows live in lanes 0..15 of each quadrant
    const int tok_in_page = w4 * 16 + lane;
    float l[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) l[c] = 0.f;
    if (tid_s < N) sm->m_ref[tid_s] = kMinusHuge;  // owner thread writes; the item barrier below orders the readers
    named_sync(1);

    const int npages = w.page_end - w.page_begin;
    for (int pg = 0; pg < npages; ++pg, ++g) {
        const int b = g & 1;
        mbar_wait(&sm->s_full[b], (g >> 1) & 1);
        tc_fence_after();
        float x[NC];
#pragma unroll
        for (int c0 = 0; c0 < NC; c0 += W)
            tmem_ldw<W>(tmem_addr(tmem, w4 * 32, kColS + b * 64 + cbase + c0), reinterpret_cast<uint32_t*>(&x[c0]));
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->s_empty[b]);

        const int page = w.page_begin + pg;
        const int key_pos = page * kPage + tok_in_page;
        const bool boundary = (page + 1) * kPage > w.n_keys;  // some row may not see every key of this page
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float v = x[c] * p.scale_log2;
            const bool ok = lane_ok && (!boundary || key_pos < w.n_keys + (N == 64 ? ((cbase + c) >> 4) : 0));
            x[c] = ok ? v : -INFINITY;
        }
        // Lazy running max: the per-row maximum is refreshed only when some key of this page exceeds the row's
        // reference by more than 2^kRescaleThreshold (always on the first page, where m_ref = -1e30).  The common
        // path costs one subtraction + max per value and a single bar.red.or over the softmax threads.
        float dmax = -INFINITY;
#pragma unroll
        for (int c = 0; c < NC; ++c) dmax = fmaxf(dmax, x[c] - sm->m_ref[cbase + c]);
        const bool need = named_or(2, dmax > kRescaleThreshold);
        if (need) {
            // exact column (query-row) max over the 64 keys of the page: warp redux, then 4 quadrants through smem
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                const float wm = warp_max(x[c]);
                if (lane == (c & 31)) sm->red[w4][cbase + c] = wm;
            }
            named_sync(1);
            if (tid_s < N) {
                const float tm = fmaxf(fmaxf(sm->red[0][tid_s], sm->red[1][tid_s]), fmaxf(sm->red[2][tid_s], sm->red[3][tid_s]));
                const float mo = sm->m_ref[tid_s];
                const float mn = fmaxf(mo, tm);
                sm->m_ref[tid_s] = mn;
                sm->alpha[tid_s] = ex2(mo - mn);  // 1 if unchanged, 0 if nothing had been visible before
            }
            named_sync(1);
            if (pg > 0) {  // O^T and l hold data relative to the old reference: rescale (rare)
                mbar_wait(&sm->pv_done[(g - 1) & 1], ((g - 1) >> 1) & 1);  // every PV issued so far has completed
                tc_fence_after();
#pragma unroll
                for (int b4 = 0; b4 < 4; ++b4)
#pragma unroll
                    for (int c0 = 0; c0 < NC; c0 += W) {
                        uint32_t r[W];
                        const uint32_t ta = tmem_addr(tmem, w4 * 32, kColO + b4 * 64 + cbase + c0);
                        tmem_ldw<W>(ta, r);
                        tmem_wait_ld();
#pragma unroll
                        for (int i = 0; i < W; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * sm->alpha[cbase + c0 + i]);
                        tmem_stw<W>(ta, r);
                    }
                tmem_wait_st();
#pragma unroll
                for (int c = 0; c < NC; ++c) l[c] *= sm->alpha[cbase + c];
            }
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float pv = ex2(x[c] - sm->m_ref[cbase + c]);
            l[c] += pv;
            x[c] = pv;
        }
        if (boundary && lane_ok && key_pos >= w.n_keys + w.n_q - 1) {
            // This key is invisible to every row of the item (a stale slot of the sequence's last page): its P^T row is 0, but
            // the PV MMA still multiplies the page's V rows, and 0 * NaN = NaN.  Zero the token's latent row in the page's
            // slots (128 B per 64-dim chunk; the 128-byte swizzle permutes inside the row) -- the S MMAs that read it as K
            // have completed (s_full), the fence below orders the stores before the PV MMAs.  Each column half takes 4 chunks.
            const PageSlots zs = page_slots<R>(g);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int ch = (sw >> 2) * 4 + c;
                uint4* dst = reinterpret_cast<uint4*>(kv + (zs.pair[ch >> 1] + (ch & 1)) * kSlotBytes + tok_in_page * 128);
#pragma unroll
                for (int j = 0; j < 8; ++j) dst[j] = make_uint4(0u, 0u, 0u, 0u);
            }
        }
        if (PK) {
            // decode-only instantiation: P as the MN-major B operand [64 keys][16 query rows x 2 B] (2 KB, SWIZZLE_32B: the 16-byte
            // chunk index is XORed with bit 2 of the row) in a buffer of its own, so that the page's RoPE slot can go back to the
            // ring as soon as the S MMAs have read it.  This thread's key row takes ONE 16-byte store for its 8 heads.
            if (g >= 2) mbar_wait(&sm->pv_done[b], ((g - 2) >> 1) & 1);  // PV of page g - 2 has read this P buffer
            if (lane_ok) {
                uint8_t* pb = kv + R * kSlotBytes + b * kDecPBytes;
                const uint32_t kk = uint32_t(tok_in_page);
                static_assert(!PK || NC == 8, "one 16-byte chunk per column half");
                *reinterpret_cast<uint4*>(pb + kk * 32u + (((uint32_t(cbase) >> 3) ^ ((kk >> 2) & 1u)) << 4)) =
                    make_uint4(pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]), pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
            }
        } else if (lane_ok) {  // P^T as the MN-major B operand: row = key, N bf16 along the row, SWIZZLE_128B
            uint8_t* ps = kv + page_slots<R>(g).rope * kSlotBytes;
#pragma unroll
            for (int j = 0; j < NC / 8; ++j) {
                uint4 v;
                v.x = pack_bf16(x[8 * j + 0], x[8 * j + 1]);
                v.y = pack_bf16(x[8 * j + 2], x[8 * j + 3]);
                v.z = pack_bf16(x[8 * j + 4], x[8 * j + 5]);
                v.w = pack_bf16(x[8 * j + 6], x[8 * j + 7]);
                *reinterpret_cast<uint4*>(ps + sw128_offset(tok_in_page, cbase / 8 + j)) = v;
            }
        }
        fence_proxy_async_smem();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->p_full[b]);
    }

    // ---- epilogue: all PV MMAs of the item are complete
    mbar_wait(&sm->o_full, it & 1);
    tc_fence_after();
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        float v = l[c];
        v += __shfl_xor_sync(0xffffffffu, v, 8);
        v += __shfl_xor_sync(0xffffffffu, v, 4);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        v += __shfl_xor_sync(0xffffffffu, v, 1);  // lanes 0..15 hold the data, lanes 16..31 hold zeros
        if (lane == (c & 15)) sm->red[w4][cbase + c] = v;
    }
    named_sync(1);
    const bool is_final = w.partial_slot < 0;
    if (tid_s < N) {
        const float L = sm->red[0][tid_s] + sm->red[1][tid_s] + sm->red[2][tid_s] + sm->red[3][tid_s];
        sm->linv[tid_s] = 1.f / L;
        const float m = sm->m_ref[tid_s];
        const int tok = tid_s >> 4, h = tid_s & 15;
        if (tok < w.n_q) {
            if (is_final) {
                float* lse = w.kind ? p.lse_chunk : p.lse_dec;
                if (lse) lse[size_t(w.q_index + tok) * kHeads + h] = (m + log2f(L)) * kLn2;
            } else {
                float* ml = reinterpret_cast<float*>(p.partials + size_t(w.partial_slot + tok) * kPartialSlotBytes +
                                                     size_t(kHeads) * kLatent * 4);
                ml[h] = m;
                ml[kHeads + h] = L;
            }
        }
    }
    named_sync(2);
    // TMEM reads run at 64 B/clk per SM and each tcgen05.ld round trip costs several hundred cycles: the loads of block
    // b4 + 1 are in flight while block b4 is converted and stored
    uint32_t rr[2][NC];
    auto load_block = [&](int b4, uint32_t* r) {
#pragma unroll
        for (int c0 = 0; c0 < NC; c0 += W) tmem_ldw<W>(tmem_addr(tmem, w4 * 32, kColO + b4 * 64 + cbase + c0), r + c0);
    };
    load_block(0, rr[0]);
#pragma unroll
    for (int b4 = 0; b4 < 4; ++b4) {
        tmem_wait_ld();
        if (b4 < 3) load_block(b4 + 1, rr[(b4 + 1) & 1]);
        const uint32_t* r = rr[b4 & 1];
        const int d = b4 * 128 + w4 * 32 + lane;
#pragma unroll
        for (int c0 = 0; c0 < NC; c0 += W) {
            const int col = cbase + c0;
            const int tok = col >> 4;
            if (tok >= w.n_q) continue;  // ragged chunk tail (uniform across the warp)
            if (is_final) {
                __nv_bfloat16* o = (w.kind ? p.out_chunk : p.out_dec) + (size_t(w.q_index + tok) * kHeads + (col & 15)) * kLatent + d;
#pragma unroll
                for (int i = 0; i < W; ++i) o[i * kLatent] = __float2bfloat16_rn(__uint_as_float(r[c0 + i]) * sm->linv[col + i]);
            } else {
                float* o = reinterpret_cast<float*>(p.partials + size_t(w.partial_slot + tok) * kPartialSlotBytes) + (col & 15) * kLatent + d;
#pragma unroll
                for (int i = 0; i < W; ++i) st_f32_evict_last(o + i * kLatent, __uint_as_float(r[c0 + i]));
            }
        }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->o_empty);
}

// ------------------------------------------------------------------------------------------------------------
// MMA issue for one work item: two issuing warps (each converged, one elected lane issues).  A tcgen05.mma of these
// shapes costs its issuing warp 25-60 cycles, more than the tensor pipe needs to execute it, and an mbarrier wait ~100
// even when complete: with ONE warp the 36 S MMAs and the 16 PV MMAs of a page serialise (~2000 cycles per page) and a
// PV whose P^T is ready queues behind the S burst of the next page -- which lengthens the time a page holds its ring
// slots, and with it the bytes in flight per SM.  The S warp and the PV warp only meet through the barriers the softmax
// warps sit between (s_full -> p_full), so they run independently: S(g + 1) is issued while PV(g) is.
// tcgen05.commit tracks the issuing thread's own MMAs: the page's slots are released by the PV warp (S(g) completed
// before the softmax of page g started, i.e. before PV(g) was issued).
// ------------------------------------------------------------------------------------------------------------
template <int N, int R, bool PK>
__device__ __forceinline__ void s_item(Small* sm, uint32_t tmem, uint32_t q_base, uint32_t kv_base, int npages, uint32_t g0,
                                       uint32_t qbuf, uint32_t qfull_parity) {
    constexpr uint32_t idesc_s = make_idesc_bf16(64, N, 0, 0);   // S^T = K Q^T : A K-major, B K-major
    constexpr uint32_t desc_hi = smem_desc_hi(1024);
    const uint32_t qb_lo = smem_desc_lo(q_base, 16);
    mbar_wait(&sm->q_full[qbuf], qfull_parity);
    for (int s = 0; s < npages; ++s) {
        const uint32_t gg = g0 + s;
        const uint32_t st = gg & 1;
        mbar_wait(&sm->s_empty[st], ((gg >> 1) & 1) ^ 1);  // the softmax warps have read S^T of page gg - 2 out of this buffer
        // The page lands box by box (4 pairs of latent chunks + the RoPE chunk): the MMAs of a box are issued as soon as it is
        // there, so that S^T completes ~300 cycles after the last box instead of a whole issue burst (~1270) later.  This warp
        // has nothing else to do meanwhile.
        const PageSlots ps = page_slots<R>(gg);
        uint64_t* full = sm->kv_full[gg & (kPageRing - 1)];
        const uint32_t par = (gg / kPageRing) & 1;
        auto chunk_mmas = [&](uint32_t c, uint32_t slot, bool first) {
            const uint32_t ka_lo = smem_desc_lo(kv_base + slot * kSlotBytes, 16);
#pragma unroll
            for (uint32_t j = 0; j < 4; ++j)
                umma_bf16_ss_lohi(tmem + kColS + st * 64, ka_lo + ((j * 32) >> 4), desc_hi,
                                  qb_lo + ((c * N * 128 + j * 32) >> 4), desc_hi, idesc_s, !(first && j == 0));
        };
        // Fixed accumulation order (latent chunks 0..7, then the RoPE chunk) whatever the page's slot parity: the order of
        // the fp32 partial sums must not depend on which pages a CTA happened to pop (results are bit-reproducible).
#pragma unroll
        for (uint32_t b = 0; b < 4; ++b) {
            mbar_wait(&full[b], par);
            tc_fence_after();
            chunk_mmas(2 * b, ps.pair[b], b == 0);
            chunk_mmas(2 * b + 1, ps.pair[b] + 1, false);
        }
        mbar_wait(&full[4], par);
        tc_fence_after();
        chunk_mmas(8, ps.rope, false);
        umma_commit_elect(&sm->s_full[st]);
        if (PK) umma_commit_elect(&sm->kv_empty[gg & (kPageRing - 1)][4]);  // the RoPE slot is only ever read by these MMAs
        if (s == npages - 1) {  // Q buffer(s) free once every S-MMA retires
            umma_commit_elect(&sm->q_empty[qbuf]);
            if (N == 64) umma_commit_elect(&sm->q_empty[1]);
        }
    }
}

template <int N, int R, bool PK>
__device__ __forceinline__ void pv_item(Small* sm, uint32_t tmem, uint32_t kv_base, int npages, uint32_t g0, uint32_t it) {
    // O^T += V^T P^T : A = the page's latent slots MN-major; B = P, MN-major in the page's RoPE slot (SWIZZLE_128B), or (PK) in its own
    // 2 KB buffer (SWIZZLE_32B)
    constexpr uint32_t idesc_o = make_idesc_bf16(128, N, 1, 1);
    constexpr uint32_t desc_hi = smem_desc_hi(1024);
    constexpr uint32_t pdesc_hi = PK ? smem_desc_hi_sw32(256) : desc_hi;  // PK: P in atoms of 8 key rows x 32 B
    for (int pv = 0; pv < npages; ++pv) {
        const uint32_t gg = g0 + pv;
        const uint32_t pst = gg & 1, pph = (gg >> 1) & 1;
        mbar_wait(&sm->p_full[pst], pph);
        if (pv == 0) mbar_wait(&sm->o_empty, (it & 1) ^ 1);  // previous item's epilogue has drained O^T
        tc_fence_after();
        const PageSlots ps = page_slots<R>(gg);
        uint64_t* empty = sm->kv_empty[gg & (kPageRing - 1)];
        const uint32_t pb_lo = PK ? smem_desc_lo(kv_base + R * kSlotBytes + pst * kDecPBytes, 16)
                                  : smem_desc_lo(kv_base + ps.rope * kSlotBytes, 8192);
#pragma unroll
        for (uint32_t b4 = 0; b4 < 4; ++b4) {
            const uint32_t va_lo = smem_desc_lo(kv_base + ps.pair[b4] * kSlotBytes, 8192);
#pragma unroll
            for (uint32_t ks = 0; ks < 4; ++ks)
                umma_bf16_ss_lohi(tmem + kColO + b4 * 64, va_lo + ((ks * 2048) >> 4), desc_hi,
                                  pb_lo + ((PK ? ks * 512 : ks * 2048) >> 4), pdesc_hi, idesc_o, (pv > 0 || ks > 0));
            umma_commit_elect(&empty[b4]);  // slot pair b4 goes back to the ring when this block's MMAs retire
        }
        if (!PK) umma_commit_elect(&empty[4]);  // P^T sat in the RoPE slot
        umma_commit_elect(&sm->pv_done[pst]);
        if (pv == npages - 1) umma_commit_elect(&sm->o_full);
    }
}

// ------------------------------------------------------------------------------------------------------------
template <bool DEC>
__global__ void __launch_bounds__(kThreads, 1)
kairos_mixed_kernel(const __grid_constant__ CUtensorMap pool_map2, const __grid_constant__ CUtensorMap pool_map1,
                    const __grid_constant__ CUtensorMap qd_map, const __grid_constant__ CUtensorMap qc_map, const KParams p) {
    using G = Geo<DEC>;
    constexpr int R = G::kSlots;
    constexpr int kOffKV = G::kOffKV;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    Small* sm = reinterpret_cast<Small*>(base + G::kOffSmall);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < 2; ++i) {
            mbar_init(&sm->q_full[i], 1);
            mbar_init(&sm->q_empty[i], 1);
        }
        for (int i = 0; i < kPageRing; ++i) {
            for (int bx = 0; bx < 5; ++bx) mbar_init(&sm->kv_full[i][bx], 1);
            for (int bx = 0; bx < 5; ++bx) mbar_init(&sm->kv_empty[i][bx], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&sm->s_full[i], 1);
            mbar_init(&sm->s_empty[i], kSoftmaxWarps);
            mbar_init(&sm->item_full[i], 1);
            mbar_init(&sm->item_empty[i], 2 + kSoftmaxWarps);
            mbar_init(&sm->p_full[i], kSoftmaxWarps);
            mbar_init(&sm->pv_done[i], 1);
        }
        mbar_init(&sm->o_full, 1);
        mbar_init(&sm->o_empty, kSoftmaxWarps);
        fence_barrier_init();
    }
    if (warp == 0 && lane == 0) {
        prefetch_tensormap(&pool_map2);
        prefetch_tensormap(&pool_map1);
        prefetch_tensormap(&qd_map);
        prefetch_tensormap(&qc_map);
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the combine grid may pre-launch; it waits on griddepcontrol.wait
    if (warp == 1) tmem_alloc(&sm->tmem_base, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm->tmem_base;

    if (warp == 0) {
        // ================= producer: pop work items, TMA-load Q tiles and KV pages =================
        uint32_t g = 0;        // pages issued so far
        uint32_t g_acked = 0, k_acked = 0;  // release cursor: page, and group within it (kv_empty observed so far)
        int free_slots = R;
        uint32_t q_use0 = 0, q_use1 = 0;  // how many items have used each Q buffer (a chunk tile uses both)
        const uint32_t kv_u32 = smem_u32(base + kOffKV);
        for (uint32_t it = 0;; ++it) {
            int idx = int(blockIdx.x);  // the first item is static (grid <= n_items): no queue round trip before the first load
            if (it > 0 || !p.static_first) {
                if (lane == 0) idx = atomicAdd(&p.counters[0], 1) + (p.static_first ? int(gridDim.x) : 0);
                idx = __shfl_sync(0xffffffffu, idx, 0);
            }
            if (idx >= p.n_items) idx = -1;
            if (lane == 0) {
                mbar_wait(&sm->item_empty[it & 1], ((it >> 1) & 1) ^ 1);
                sm->item_ring[it & 1] = idx;
                mbar_arrive(&sm->item_full[it & 1]);
            }
            if (idx < 0) break;
            const WorkItem w = load_item(p.items + idx);
            const int N = (!DEC && w.kind) ? 64 : 16;
            const bool is_chunk = !DEC && w.kind;
            const int qb = is_chunk ? 0 : int(it & 1);
            if (lane == 0) {
                mbar_wait(&sm->q_empty[qb], ((qb ? q_use1 : q_use0) & 1) ^ 1);
                if (is_chunk) mbar_wait(&sm->q_empty[1], (q_use1 & 1) ^ 1);
                mbar_arrive_expect_tx(&sm->q_full[qb], uint32_t(9 * N * 128));
                const CUtensorMap* qm = is_chunk ? &qc_map : &qd_map;
                for (int c = 0; c < 9; ++c)
                    tma_load_2d(base + kOffQ + qb * kDecQBytes + c * N * 128, qm, &sm->q_full[qb], c * 64, w.q_index * kHeads, kEvictFirst);
            }
            if (qb == 0) ++q_use0;
            if (qb == 1 || is_chunk) ++q_use1;
            const int32_t* pt = (w.kind ? p.chunk_pt : p.dec_pt + size_t(w.q_index) * p.dec_stride) + w.page_begin;
            const uint64_t policy = w.kind ? kEvictLast : kEvictFirst;  // chunk KV is re-read by every tile
            const int npages = w.page_end - w.page_begin;
            for (int i = 0; i < npages; i += 32) {
                const int my = (i + lane < npages) ? __ldg(pt + i + lane) : 0;
                const int cnt = min(32, npages - i);
                for (int j = 0; j < cnt; ++j, ++g) {
                    const int pid = __shfl_sync(0xffffffffu, my, j);
                    if (lane == 0) {
                        const PageSlots ps = page_slots<R>(g);
                        uint64_t* full = sm->kv_full[g & (kPageRing - 1)];  // one barrier per box: [0..3] latent pairs, [4] RoPE chunk
                        const int row = pid * kPage;
                        // take slots in ring order; pages retire in order, 9 slots each
                        // Slots come back group by group (the page's RoPE slot and its 4 slot pairs), in ring order: for a page
                        // that starts at an odd slot the RoPE slot is first, else last.
                        auto reserve = [&](int n) {
                            while (free_slots < n) {
                                const uint32_t odd = ((g_acked * 9u) % uint32_t(R)) & 1u;
                                const uint32_t grp = odd ? (k_acked == 0 ? 4u : k_acked - 1u) : k_acked;
                                mbar_wait(&sm->kv_empty[g_acked & (kPageRing - 1)][grp], (g_acked / kPageRing) & 1);
                                free_slots += grp == 4 ? 1 : 2;
                                if (++k_acked == 5) { k_acked = 0; ++g_acked; }
                            }
                            free_slots -= n;
                        };
                        if (ps.odd) {
                            reserve(1);
                            mbar_arrive_expect_tx(&full[4], kSlotBytes);
                            tma_load_chunks(kv_u32 + ps.rope * kSlotBytes, &pool_map1, &full[4], row, 8, policy);
                        }
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            reserve(2);
                            mbar_arrive_expect_tx(&full[b], 2 * kSlotBytes);
                            tma_load_chunks(kv_u32 + ps.pair[b] * kSlotBytes, &pool_map2, &full[b], row, 2 * b, policy);
                        }
                        if (!ps.odd) {
                            reserve(1);
                            mbar_arrive_expect_tx(&full[4], kSlotBytes);
                            tma_load_chunks(kv_u32 + ps.rope * kSlotBytes, &pool_map1, &full[4], row, 8, policy);
                        }
                    }
                }
            }
        }
    } else if (warp == 1 || warp == kPvWarp) {
        // ================= MMA issuers: warp 1 issues the S MMAs, warp kPvWarp the PV MMAs (each converged, one elected lane)
        const uint32_t q_base = smem_u32(base + kOffQ), kv_base = smem_u32(base + kOffKV);
        uint32_t q_full0 = 0, q_full1 = 0;
        uint32_t g = 0;
        for (uint32_t it = 0;; ++it) {
            mbar_wait(&sm->item_full[it & 1], (it >> 1) & 1);
            const int idx = __shfl_sync(0xffffffffu, sm->item_ring[it & 1], 0);
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->item_empty[it & 1]);
            __syncwarp();
            if (idx < 0) break;
            const WorkItem w = load_item(p.items + idx);
            const int kind = __shfl_sync(0xffffffffu, w.kind, 0);
            const int npages = __shfl_sync(0xffffffffu, w.page_end - w.page_begin, 0);
            const bool chunk = !DEC && kind;
            if (warp == 1) {
                // Q buffer bookkeeping mirrors the producer's: q_full[b] completes once per item that loads into buffer b
                const uint32_t qb = chunk ? 0u : (it & 1u);
                const uint32_t qpar = (qb ? q_full1 : q_full0) & 1u;
                if (qb) ++q_full1; else ++q_full0;
                if (chunk) s_item<64, R, false>(sm, tmem, q_base, kv_base, npages, g, 0, qpar);
                else s_item<16, R, DEC>(sm, tmem, q_base + qb * kDecQBytes, kv_base, npages, g, qb, qpar);
            } else {
                if (chunk) pv_item<64, R, false>(sm, tmem, kv_base, npages, g, it);
                else pv_item<16, R, DEC>(sm, tmem, kv_base, npages, g, it);
            }
            g += npages;
        }
    } else {
        // ================= softmax / correction / epilogue warps =================
        const int sw = warp - 2;  // 0..7; TMEM lane quadrant = warp & 3 = (sw + 2) & 3
        uint8_t* kv = base + kOffKV;
        uint32_t g = 0;
        for (uint32_t it = 0;; ++it) {
            mbar_wait(&sm->item_full[it & 1], (it >> 1) & 1);
            const int idx = sm->item_ring[it & 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->item_empty[it & 1]);
            if (idx < 0) break;
            const WorkItem w = load_item(p.items + idx);
            if (!DEC && w.kind) softmax_item<64, R, false>(sm, kv, w, p, tmem, sw, lane, g, it);
            else softmax_item<16, R, DEC>(sm, kv, w, p, tmem, sw, lane, g, it);
        }
    }

    // ---- teardown
    tc_fence_before();
    __syncthreads();
    // When this grid was launched behind the pair kernel with programmatic stream serialisation it never waited for it; it
    // does so before it exits, so that "this grid has completed" implies "the pair grid has completed" for everything that
    // follows in the stream (the combine, the caller's consumers of out_chunk).  No-op for an ordinary launch.
    if (threadIdx.x == 0) asm volatile("griddepcontrol.wait;" ::: "memory");
    if (warp == 1) tmem_dealloc(tmem, kTmemCols);
    if (threadIdx.x == 0) {
        __threadfence();
        const int prev = atomicAdd(&p.counters[1], 1);
        if (prev == int(gridDim.x) - 1) {  // last CTA out re-arms the queue for the next launch (stream-ordered)
            p.counters[0] = 0;
            p.counters[1] = 0;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// a5: log-sum-exp combine of split partials: out = sum_k 2^(m_k-m*) O_k / sum_k 2^(m_k-m*) l_k
// grid = (combine items, kCombineSlices): each CTA merges a 32-wide slice of the 512 latent dims for all 16 heads,
// so that one long request (many splits) is spread over 16 CTAs and every thread streams independent float4 loads.
// Launched with programmatic stream serialisation: griddepcontrol.wait orders it after the main kernel's writes.
// ------------------------------------------------------------------------------------------------------------
constexpr int kCombineSlices = 16;
constexpr int kCombineThreads = 128;
__global__ void __launch_bounds__(kCombineThreads) combine_kernel(const CombineItem* __restrict__ items, const uint8_t* __restrict__ partials,
                                                      __nv_bfloat16* __restrict__ out_dec, __nv_bfloat16* __restrict__ out_chunk,
                                                      float* __restrict__ lse_dec, float* __restrict__ lse_chunk) {
    constexpr int kMaxK = 64;  // splits whose weights are staged in shared memory per pass
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the next step's append may pre-launch (it waits for this grid)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const CombineItem ci = items[blockIdx.x];
    const int kind = ci.kind_stride & 0xff, stride = ci.kind_stride >> 8;
    __shared__ float s_w[kMaxK][kHeads], s_wl[kMaxK][kHeads], s_mstar[kHeads], s_L[kHeads];
    const int tid = threadIdx.x;
    auto slot_ptr = [&](int k) { return partials + size_t(ci.first_slot + k * stride) * kPartialSlotBytes; };
    auto ml_ptr = [&](int k) { return reinterpret_cast<const float*>(slot_ptr(k) + size_t(kHeads) * kLatent * 4); };
    // the first kPre splits' data are requested before the (dependent) weight passes, so their latency overlaps
    constexpr int kPre = 8;
    const int fo_pre = ((tid >> 3) * kLatent + blockIdx.y * 32 + (tid & 7) * 4) / 4;
    float4 pre[kPre];
#pragma unroll
    for (int k = 0; k < kPre; ++k)
        pre[k] = k < ci.n_splits ? __ldcs(reinterpret_cast<const float4*>(slot_ptr(k)) + fo_pre) : make_float4(0.f, 0.f, 0.f, 0.f);
    // pass 1: m* per head over all splits (8 parts x 16 heads)
    {
        const int h = tid & 15, part = tid >> 4;  // 8 parts
        float ms = kMinusHuge;
        for (int k = part; k < ci.n_splits; k += 8) ms = fmaxf(ms, ml_ptr(k)[h]);
        __shared__ float s_pm[8][kHeads];
        s_pm[part][h] = ms;
        __syncthreads();
        if (tid < kHeads) {
            float m2 = kMinusHuge;
#pragma unroll
            for (int i = 0; i < 8; ++i) m2 = fmaxf(m2, s_pm[i][tid]);
            s_mstar[tid] = m2;
            s_L[tid] = 0.f;
        }
        __syncthreads();
    }
    // thread -> (head h, 4 consecutive dims of this CTA's 32-dim slice)
    const int h = tid >> 3;
    const int d0 = blockIdx.y * 32 + (tid & 7) * 4;
    const int fo = (h * kLatent + d0) / 4;  // float4 index inside a slot
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k0 = 0; k0 < ci.n_splits; k0 += kMaxK) {
        const int kn = min(kMaxK, ci.n_splits - k0);
        for (int i = tid; i < kn * kHeads; i += kCombineThreads) {
            const int k = i / kHeads, hh = i % kHeads;
            const float* ml = ml_ptr(k0 + k);
            const float w = exp2f(ml[hh] - s_mstar[hh]);  // m = -1e30 (nothing visible) -> 0
            s_w[k][hh] = w;
            s_wl[k][hh] = w * ml[kHeads + hh];
        }
        __syncthreads();
        if (tid < kHeads) {  // deterministic order: the result must not depend on scheduling
            float Ls = s_L[tid];
            for (int k = 0; k < kn; ++k) Ls += s_wl[k][tid];
            s_L[tid] = Ls;
        }
        int kb = 0;
        if (k0 == 0) {
#pragma unroll
            for (int k = 0; k < kPre; ++k) {
                const float w = k < kn ? s_w[k][h] : 0.f;
                acc[0] += w * pre[k].x; acc[1] += w * pre[k].y; acc[2] += w * pre[k].z; acc[3] += w * pre[k].w;
            }
            kb = kPre;
        }
#pragma unroll 8
        for (int k = kb; k < kn; ++k) {
            const float4 a = __ldcs(reinterpret_cast<const float4*>(slot_ptr(k0 + k)) + fo);  // streamed: read once
            const float w = s_w[k][h];
            acc[0] += w * a.x; acc[1] += w * a.y; acc[2] += w * a.z; acc[3] += w * a.w;
        }
        __syncthreads();
    }
    const float L = s_L[h];
    if (blockIdx.y == 0 && tid < kHeads) {
        float* lse = kind ? lse_chunk : lse_dec;
        if (lse) lse[size_t(ci.q_index) * kHeads + tid] = (s_mstar[tid] + log2f(s_L[tid])) * kLn2;
    }
    const float inv = 1.f / L;
    __nv_bfloat16* out = (kind ? out_chunk : out_dec) + (size_t(ci.q_index) * kHeads + h) * kLatent + d0;
    uint2 o;
    o.x = pack_bf16(acc[0] * inv, acc[1] * inv);
    o.y = pack_bf16(acc[2] * inv, acc[3] * inv);
    *reinterpret_cast<uint2*>(out) = o;
}

// ------------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

// ------------------------------------------------------------------------------------------------------------
// kairos_decode_static: decode attention with NO allocation anywhere (include/kairos.h).  Everything the split-KV decode needs
// beyond the caller's inputs and outputs -- the work-queue counters, the work list, the combine list and the fp32 split partials --
// lives in this file-scope array, which every GPU that loads the library holds until the process exits (about 9.3 MiB).
// In HOST code the name `g_static_scratch` is a host-side stand-in, not a device address: umma_init asks cudaGetSymbolAddress for
// the real one, once per device with that device current, and the launches below are given that pointer.  Device code may name
// the array directly (static_plan_kernel does).  Every call on a device shares the array and it keeps the last call's contents:
// the plan kernel clears the counters and rewrites both lists at the start of every call; calls that overlap on the GPU race.
// ------------------------------------------------------------------------------------------------------------
constexpr int kStaticMaxDecodes = KAIROS_STATIC_MAX_DECODES;  // 128
constexpr int kStaticTargetPieces = 148;                       // a request longer than total_pages / 148 (min 4 pages) is split
constexpr int kStaticMaxSlots = 2 * kStaticTargetPieces;       // split pieces <= total/per + #split requests <= 2 * 148
constexpr int kStaticMaxItems = kStaticMaxDecodes + kStaticMaxSlots;
constexpr size_t kStaticOffItems = 256;                        // [0, 256): queue counters
constexpr size_t kStaticOffCombines = kStaticOffItems + size_t(kStaticMaxItems) * sizeof(WorkItem);
constexpr size_t kStaticOffPartials = (kStaticOffCombines + size_t(kStaticMaxDecodes) * sizeof(CombineItem) + 255) / 256 * 256;
constexpr size_t kStaticScratchBytes = kStaticOffPartials + size_t(kStaticMaxSlots) * kPartialSlotBytes;
static __device__ __align__(256) uint8_t g_static_scratch[kStaticScratchBytes];
uint8_t* g_static_ptr[64] = {};  // device address of g_static_scratch per device ordinal (filled by umma_init)

struct StaticLens {
    int32_t v[kStaticMaxDecodes];
};

// pages per piece for a step with `total_pages` pages in all: the ONE rule both the host (grid sizes) and the device (lists) apply
__host__ __device__ inline int32_t static_piece_pages(int64_t total_pages) {
    const int64_t per = (total_pages + kStaticTargetPieces - 1) / kStaticTargetPieces;
    return int32_t(per < 4 ? 4 : per);
}

// One block: request i = thread i.  Clears the counters, writes the work list (request order, pieces of `per` pages) and the combine
// list (one entry per request that was split) into g_static_scratch.
__global__ void __launch_bounds__(kStaticMaxDecodes) static_plan_kernel(const StaticLens lens, int32_t n_dec, int32_t per) {
    __shared__ int32_t s_item0[kStaticMaxDecodes + 1], s_slot0[kStaticMaxDecodes + 1], s_comb0[kStaticMaxDecodes + 1];
    const int i = threadIdx.x;
    if (i < 64) reinterpret_cast<int32_t*>(g_static_scratch)[i] = 0;  // queue counters: must start at zero
    const int32_t pages = i < n_dec ? (lens.v[i] + kPage - 1) / kPage : 0;
    const int32_t n_splits = i < n_dec ? max(1, (pages + per - 1) / per) : 0;
    s_item0[i + 1] = n_splits;
    s_slot0[i + 1] = n_splits > 1 ? n_splits : 0;
    s_comb0[i + 1] = n_splits > 1 ? 1 : 0;
    __syncthreads();
    if (i == 0) {
        s_item0[0] = s_slot0[0] = s_comb0[0] = 0;
        for (int k = 1; k <= n_dec; ++k) {
            s_item0[k] += s_item0[k - 1];
            s_slot0[k] += s_slot0[k - 1];
            s_comb0[k] += s_comb0[k - 1];
        }
    }
    __syncthreads();
    if (i >= n_dec) return;
    WorkItem* items = reinterpret_cast<WorkItem*>(g_static_scratch + kStaticOffItems);
    CombineItem* combines = reinterpret_cast<CombineItem*>(g_static_scratch + kStaticOffCombines);
    for (int32_t sp = 0; sp < n_splits; ++sp) {
        WorkItem w;
        w.kind = 0;
        w.q_index = i;
        w.page_begin = sp * per;
        w.page_end = min(pages, (sp + 1) * per);
        w.n_keys = lens.v[i];
        w.n_q = 1;
        w.partial_slot = n_splits > 1 ? s_slot0[i] + sp : -1;
        w.cost = 0;
        items[s_item0[i] + sp] = w;
    }
    if (n_splits > 1) combines[s_comb0[i]] = CombineItem{i, s_slot0[i], n_splits, 0 /*decode*/ | (1 << 8) /*slot stride 1*/};
}

}  // namespace

int umma_chunk_tile_tokens() { return kChunkTileTokens; }
int umma_resident_ctas(const kairos_ctx* ctx) { return ctx->sm_count; }

// q viewed as [rows][576] bf16 with boxes of 64 dims x box_rows rows.  cuTensorMapEncodeTiled costs a few microseconds of
// host time, so the encoded map is kept while the caller passes the same buffer.
int encode_q_map(QMapCache* cache, const void* ptr, uint64_t rows, uint32_t box_rows) {
    return encode_2d_map(cache, ptr, kDim, rows, kTokenBytes, 64, box_rows);
}

int encode_2d_map(QMapCache* cache, const void* ptr, uint64_t inner, uint64_t rows, uint64_t row_stride_bytes, uint32_t box_inner,
                  uint32_t box_rows) {
    if (cache->ptr == ptr && cache->rows == rows) return KAIROS_OK;
    cuuint64_t dims[2] = {cuuint64_t(inner), rows};
    cuuint64_t strides[1] = {cuuint64_t(row_stride_bytes)};
    cuuint32_t box[2] = {box_inner, box_rows};
    cuuint32_t es[2] = {1, 1};
    CUresult r = g_encode(&cache->map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, es,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        cache->ptr = nullptr;
        return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled failed: " + std::to_string(int(r)));
    }
    cache->ptr = ptr;
    cache->rows = rows;
    return KAIROS_OK;
}

int encode_tiled_map(CUtensorMap* out, bool u8, int rank, const void* ptr, const uint64_t* dims, const uint64_t* strides, const uint32_t* box) {
    if (!g_encode) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled not available");
    cuuint64_t d[3], st[2];
    cuuint32_t bx[3], es[3] = {1, 1, 1};
    for (int i = 0; i < rank; ++i) { d[i] = dims[i]; bx[i] = box[i]; }
    for (int i = 0; i + 1 < rank; ++i) st[i] = strides[i];
    const CUresult r = g_encode(out, u8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, cuuint32_t(rank),
                                const_cast<void*>(ptr), d, st, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled failed: " + std::to_string(int(r)));
    return KAIROS_OK;
}

int umma_init(kairos_ctx* ctx) {
    if (!g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        KAIROS_CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled not available");
        g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    }
    // pool viewed as [chunk 9][row num_pages*64][64 elems]: one box = one page as [9][64][128 B]
    cuuint64_t dims[3] = {64, cuuint64_t(ctx->cfg.num_pages) * kPage, 9};
    cuuint64_t strides[2] = {cuuint64_t(kTokenBytes), 128};
    cuuint32_t box[3] = {64, 64, 9};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = g_encode(&ctx->pool_map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, ctx->cfg.pool, dims, strides, box, es,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled(pool) failed: " + std::to_string(int(r)));
    // the ring is filled by boxes of 2 latent chunks (16 KB) and 1 RoPE chunk (8 KB)
    for (int n = 1; n <= 2; ++n) {
        cuuint32_t boxn[3] = {64, 64, cuuint32_t(n)};
        r = g_encode(n == 2 ? &ctx->pool_map2 : &ctx->pool_map1, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, ctx->cfg.pool, dims, strides, boxn,
                     es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(KAIROS_ERR_CUDA, "cuTensorMapEncodeTiled(pool chunks) failed: " + std::to_string(int(r)));
    }
    KAIROS_CUDA_TRY(cudaFuncSetAttribute(kairos_mixed_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, Geo<false>::kSmemBytes));
    KAIROS_CUDA_TRY(cudaFuncSetAttribute(kairos_mixed_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, Geo<true>::kSmemBytes));
    KAIROS_CUDA_TRY(cudaMemset(ctx->cfg.workspace, 0, 256));  // work-queue counters
    // kairos_decode_static: the device address of the file-scope scratch, once per device, with that device current (kairos_create
    // has made it so).  The host-side name of a __device__ array must never be handed to a kernel.
    const int dev = ctx->cfg.device;
    if (dev >= 0 && dev < 64 && !g_static_ptr[dev]) {
        void* ptr = nullptr;
        KAIROS_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_scratch));
        g_static_ptr[dev] = static_cast<uint8_t*>(ptr);
    }
    return KAIROS_OK;
}

int launch_attn_umma(kairos_ctx* ctx, const Plan& plan, const StepArgs& a, const WorkItem* dev_items, int32_t n_items,
                     cudaStream_t stream, int max_ctas, bool as_clusters, bool pdl) {
    // placeholders when a side is empty (never dereferenced); the caller has encoded the maps the step needs
    const CUtensorMap& qd_map = a.n_dec > 0 ? ctx->qd_map.map : ctx->pool_map;
    const CUtensorMap& qc_map = (a.chunk_len > 0 && plan.n_chunk_items > 0) ? ctx->qc_map.map : ctx->pool_map;
    KParams p;
    p.items = dev_items;
    p.n_items = n_items;
    p.counters = reinterpret_cast<int32_t*>(ctx->cfg.workspace);
    p.dec_pt = a.dec_page_tables;
    p.dec_stride = a.dec_table_stride;
    p.chunk_pt = a.chunk_page_table;
    p.out_dec = reinterpret_cast<__nv_bfloat16*>(a.out_dec);
    p.out_chunk = reinterpret_cast<__nv_bfloat16*>(a.out_chunk);
    p.lse_dec = a.lse_dec;
    p.lse_chunk = a.lse_chunk;
    p.partials = reinterpret_cast<uint8_t*>(ctx->cfg.workspace) + 256;
    p.scale_log2 = ctx->cfg.softmax_scale * 1.4426950408889634f;
    int grid = std::max(1, std::min(n_items, std::min(max_ctas, umma_resident_ctas(ctx))));
    // beside the pair kernel the grid is launched as 2-CTA clusters (nothing in the kernel uses the cluster): it then
    // occupies whole TPCs, which the chunk clusters need, and the first item comes from the queue (a CTA that becomes
    // resident late must not be holding a statically assigned item)
    const bool with_pairs = plan.n_pairs > 0;
    if (as_clusters) grid = std::max(2, std::min(max_ctas, umma_resident_ctas(ctx)) & ~1);
    p.static_first = with_pairs ? 0 : 1;
    // decode-only queues (no chunk, or the chunk is on the pair grid) take the instantiation with the deeper page ring
    bool dec_only = a.chunk_len == 0 || plan.n_chunk_items == 0;
    if (ctx->force_dec_only >= 0) dec_only = dec_only && ctx->force_dec_only != 0;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(grid), 1, 1);
    cfg.blockDim = dim3(kThreads, 1, 1);
    cfg.dynamicSmemBytes = dec_only ? Geo<true>::kSmemBytes : Geo<false>::kSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[2];
    int n_attr = 0;
    if (as_clusters) {
        attr[n_attr].id = cudaLaunchAttributeClusterDimension;
        attr[n_attr].val.clusterDim.x = 2;
        attr[n_attr].val.clusterDim.y = 1;
        attr[n_attr].val.clusterDim.z = 1;
        ++n_attr;
    }
    if (pdl) {  // queued behind the pair kernel: CTAs become resident as clusters finish (this kernel never waits on it)
        attr[n_attr].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[n_attr].val.programmaticStreamSerializationAllowed = 1;
        ++n_attr;
    }
    cfg.attrs = attr;
    cfg.numAttrs = n_attr;
    if (dec_only)
        KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kairos_mixed_kernel<true>, ctx->pool_map2, ctx->pool_map1, qd_map, qc_map, p));
    else
        KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kairos_mixed_kernel<false>, ctx->pool_map2, ctx->pool_map1, qd_map, qc_map, p));
    return KAIROS_OK;
}

// a5 launch (after the attention kernels of the step; programmatic dependent launch on the preceding kernel)
int launch_combine(kairos_ctx* ctx, const StepArgs& a, const CombineItem* dev_combines, int32_t n_combines, cudaStream_t stream) {
    if (n_combines > 0) {
        const uint8_t* partials = reinterpret_cast<uint8_t*>(ctx->cfg.workspace) + 256;
        __nv_bfloat16* out_dec = reinterpret_cast<__nv_bfloat16*>(a.out_dec);
        __nv_bfloat16* out_chunk = reinterpret_cast<__nv_bfloat16*>(a.out_chunk);
        float* lse_dec = a.lse_dec;
        float* lse_chunk = a.lse_chunk;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(unsigned(n_combines), kCombineSlices, 1);
        cfg.blockDim = dim3(kCombineThreads, 1, 1);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        // with two attention kernels in flight the second one waits for the first before it exits, so following it is enough
        cfg.numAttrs = 1;
        KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, combine_kernel, dev_combines, partials, out_dec, out_chunk, lse_dec, lse_chunk));
    }
    return KAIROS_OK;
}

// kairos_decode_static (include/kairos.h): plan on the device, decode splits, LSE combine -- three launches, no allocation.
int launch_decode_static(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                         const int32_t* dec_ctx_lens, void* out_dec, float* lse_dec, cudaStream_t stream) {
    const int dev = ctx->cfg.device;
    uint8_t* scratch = (dev >= 0 && dev < 64) ? g_static_ptr[dev] : nullptr;
    if (!scratch) return fail(KAIROS_ERR_CUDA, "static scratch has no device address on this device (kairos_create looks it up)");
    if (n_dec > kStaticMaxDecodes)
        return fail(KAIROS_ERR_WORKSPACE, "kairos_decode_static takes at most " + std::to_string(kStaticMaxDecodes) + " decodes per call (got " +
                                              std::to_string(n_dec) + "): its scratch is a fixed array");
    // the same arithmetic as static_plan_kernel, for the grid sizes only
    StaticLens lens{};
    int64_t total_pages = 0;
    for (int32_t i = 0; i < n_dec; ++i) {
        lens.v[i] = dec_ctx_lens[i];
        total_pages += (dec_ctx_lens[i] + kPage - 1) / kPage;
    }
    const int32_t per = static_piece_pages(total_pages);
    int32_t n_items = 0, n_slots = 0, n_combines = 0;
    for (int32_t i = 0; i < n_dec; ++i) {
        const int32_t pages = (dec_ctx_lens[i] + kPage - 1) / kPage;
        const int32_t n_splits = std::max(1, (pages + per - 1) / per);
        n_items += n_splits;
        if (n_splits > 1) {
            n_slots += n_splits;
            ++n_combines;
        }
    }
    if (n_items > kStaticMaxItems || n_slots > kStaticMaxSlots)
        return fail(KAIROS_ERR_WORKSPACE, "kairos_decode_static: the step needs more split pieces than its fixed scratch holds");
    if (int rc = encode_q_map(&ctx->qs_map, q_dec, uint64_t(n_dec) * kHeads, 16)) return rc;

    static_plan_kernel<<<1, kStaticMaxDecodes, 0, stream>>>(lens, n_dec, per);
    KAIROS_CUDA_TRY(cudaGetLastError());

    KParams p;
    p.items = reinterpret_cast<const WorkItem*>(scratch + kStaticOffItems);
    p.n_items = n_items;
    p.counters = reinterpret_cast<int32_t*>(scratch);
    p.dec_pt = dec_page_tables;
    p.dec_stride = dec_table_stride;
    p.chunk_pt = nullptr;
    p.out_dec = reinterpret_cast<__nv_bfloat16*>(out_dec);
    p.out_chunk = nullptr;
    p.lse_dec = lse_dec;
    p.lse_chunk = nullptr;
    p.partials = scratch + kStaticOffPartials;
    p.scale_log2 = ctx->cfg.softmax_scale * 1.4426950408889634f;
    p.static_first = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(std::max(1, std::min(n_items, umma_resident_ctas(ctx)))), 1, 1);
    cfg.blockDim = dim3(kThreads, 1, 1);
    cfg.dynamicSmemBytes = Geo<true>::kSmemBytes;
    cfg.stream = stream;
    cfg.attrs = nullptr;
    cfg.numAttrs = 0;
    // qc_map is a placeholder (the decode-only instantiation never reads it)
    KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kairos_mixed_kernel<true>, ctx->pool_map2, ctx->pool_map1, ctx->qs_map.map, ctx->pool_map, p));
    if (n_combines > 0) {
        const CombineItem* dev_combines = reinterpret_cast<const CombineItem*>(scratch + kStaticOffCombines);
        const uint8_t* partials = scratch + kStaticOffPartials;
        __nv_bfloat16* od = reinterpret_cast<__nv_bfloat16*>(out_dec);
        __nv_bfloat16* oc = nullptr;
        float* lc = nullptr;
        cudaLaunchConfig_t cc{};
        cc.gridDim = dim3(unsigned(n_combines), kCombineSlices, 1);
        cc.blockDim = dim3(kCombineThreads, 1, 1);
        cc.dynamicSmemBytes = 0;
        cc.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cc.attrs = attr;
        cc.numAttrs = 1;
        KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cc, combine_kernel, dev_combines, partials, od, oc, lse_dec, lc));
    }
    return KAIROS_OK;
}

}  // namespace kairos
