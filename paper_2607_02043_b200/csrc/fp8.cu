// the fp8 latent cache (include/kairos.h, G23 / 6.7) -- quantising append, query preparation
// and the decode attention kernel over e4m3 pages.
//
// A page is codes u8 [64][512] | RoPE bf16 [64][64] | scales f32 [64] (41,216 B).  The attention kernel is the decode-only
// pipeline of attn_umma.cu re-cut for 8-bit operands, with NO dequantisation pass: the tensor cores read the codes.
//
//   S8^T[64 keys x 32] = K8_page[64 x 512] . [Qhi ; Qlo]^T       tcgen05.mma kind::f8f6f4, M=64 N=32 K=32, 16 per page
//   SR^T[64 keys x 16] = KR_page[64 x 64]  . QR^T                kind::f16 (bf16), M=64 N=16 K=16, 4 per page
//   x[t,h] = ((S8hi + S8lo) * s_t / g_h + SR) * sigma*log2(e)      s_t = the token's scale, g_h = the query row's gain (2^k)
//   y = x + log2(s_t):  P8[t,h] = 2^(y - m_h), split into two e4m3 terms;  l_h += P8 / s_t   (= 2^(x - m_h))
//   O^T[512 x 32]     += V8^T[512 x 64] . [Phi ; Plo]^T           kind::f8f6f4, M=128 N=32 K=32, A and B MN-major (A = the same page)
//   out[h] = (O[:,h] + O[:,16+h]) / l_h
//
// The token scale rides the softmax weight (P8 = p * s_t), so that O accumulates real dequantised values without touching
// the codes; running the online-softmax reference on y keeps P8 inside e4m3's range whatever the scales are.  q and P enter
// as head + remainder (two e4m3 numbers, 8 significant bits together): the products are exact in the fp32 accumulator, so
// the only rounding beyond the bf16 kernel's is the 2^-8 of those two splits.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_fp8.h>

#include <algorithm>

#include "kairos_internal.h"
#include "umma_ptx.cuh"

namespace kairos {
namespace {
using namespace ptx;

constexpr int kPage8Bytes = KAIROS_FP8_PAGE_BYTES;
constexpr int kOffRope8 = kPage * kLatent;                // 32,768
constexpr int kOffScale8 = kOffRope8 + kPage * kRope * 2;  // 40,960
static_assert(kOffScale8 + kPage * 4 == kPage8Bytes, "page layout");
constexpr int kQ8Bytes = 32 * kLatent;                     // [hi 16 rows ; lo 16 rows] x 512 codes = 16 KB per request

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }
__device__ __forceinline__ uint32_t e4m3x2(float a, float b) {  // low byte = code(a), high byte = code(b)
    return uint32_t(__nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3));
}
__device__ __forceinline__ float2 e4m3x2_value(uint32_t c) {
    const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2(__nv_fp8x2_storage_t(c), __NV_E4M3);
    return __half22float2(*reinterpret_cast<const __half2*>(&h));
}

// ------------------------------------------------------------------------------------------------------------
// quantising append: one warp per token, lane L owns latent elements [16 L, 16 L + 16)
// ------------------------------------------------------------------------------------------------------------
// positions == nullptr: token j of ONE request goes to position start_pos + j through `page_table`; otherwise token j is the newest
// token of request j and goes to positions[j] through row j of `page_table` (stride table_stride).
__global__ void __launch_bounds__(256) fp8_append_kernel(uint8_t* __restrict__ pool8, const uint4* __restrict__ latent,
                                                         const uint4* __restrict__ k_rope, const int32_t* __restrict__ page_table,
                                                         int32_t n_tokens, int32_t start_pos, const int32_t* __restrict__ positions,
                                                         int32_t table_stride) {
    const int lane = threadIdx.x & 31;
    const int j = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (j >= n_tokens) return;
    const uint4 a = __ldg(latent + size_t(j) * 64 + lane * 2), b = __ldg(latent + size_t(j) * 64 + lane * 2 + 1);
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    float v[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        v[2 * i] = bf16_lo(w[i]);
        v[2 * i + 1] = bf16_hi(w[i]);
    }
    float amax = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) amax = fmaxf(amax, fabsf(v[i]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const float s = amax > 0.f ? __fdiv_rn(amax, 448.f) : 1.f;
    uint32_t c[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t lo = e4m3x2(__fdiv_rn(v[4 * i], s), __fdiv_rn(v[4 * i + 1], s));
        const uint32_t hi = e4m3x2(__fdiv_rn(v[4 * i + 2], s), __fdiv_rn(v[4 * i + 3], s));
        c[i] = lo | (hi << 16);
    }
    const int32_t pos = positions ? __ldg(positions + j) : start_pos + j;
    const int32_t* row = positions ? page_table + size_t(j) * table_stride : page_table;
    uint8_t* page = pool8 + size_t(__ldg(row + pos / kPage)) * kPage8Bytes;
    const int slot = pos % kPage;
    *reinterpret_cast<uint4*>(page + slot * kLatent + lane * 16) = make_uint4(c[0], c[1], c[2], c[3]);
    if (lane < 8) *reinterpret_cast<uint4*>(page + kOffRope8 + slot * (kRope * 2) + lane * 16) = __ldg(k_rope + size_t(j) * 8 + lane);
    if (lane == 0) *reinterpret_cast<float*>(page + kOffScale8 + slot * 4) = s;
}

// ------------------------------------------------------------------------------------------------------------
// decode attention over fp8 pages.  Warp roles: warp 0 producer, warp 1 S issuer A (latent boxes 0-1) + TMEM owner, warps 2-9
// softmax / correction, warp 10 PV issuer, warp 11 S issuer B (latent boxes 2-3 + RoPE), warps 12-15 epilogue (O^T is
// double-buffered by item parity, so an item's output is written while the next item's pages stream).  Issuing a tcgen05.mma costs its warp
// ~40 cycles and an mbarrier wait ~100 whether or not it blocks: one warp issuing the page's 20 S MMAs behind five waits was
// the longest stage of the pipeline (2,250 cycles per page, measured), so the S product is cut in two halves that accumulate
// in separate TMEM columns (summed by the softmax warps, in a fixed order) and a page has two landing barriers, not five.
// ------------------------------------------------------------------------------------------------------------
constexpr int kSoftmaxWarps = 8;
constexpr int kSoftmaxThreads = kSoftmaxWarps * 32;
constexpr int kPvWarp = 2 + kSoftmaxWarps;
constexpr int kSbWarp = kPvWarp + 1;
constexpr int kEpiWarp = kSbWarp + 1;  // 12..15: epilogue warps (TMEM lane quadrant = warp & 3)
constexpr int kThreads = 64 + kSoftmaxThreads + 64 + 128;
constexpr int kSlotBytes = 8192;      // one box: [64 tokens][128 B] = 128 latent codes, or the 64 bf16 RoPE values, SWIZZLE_128B
// Pages in flight: a page's latent boxes stay in shared memory from their TMA request until its PV product completes (~8,000
// cycles: load latency + S + the softmax chain + PV), so the page rate is that lifetime over the ring depth; four stages gave
// 2,050 cycles per page against 1,770 of HBM time.  The RoPE box is only read by the S product: it lives in a ring of its own
// (two slots, released as soon as the page's S MMAs retire), which leaves room for FIVE latent stages.
constexpr int kStages = 5;            // latent stages of 4 boxes (32 KB)
constexpr int kStageBytes = 4 * kSlotBytes;
constexpr int kRopeSlots = 2;
constexpr int kQBufBytes = kQ8Bytes + 16 * kRope * 2;  // 18,432: q8 (4 boxes of [32 rows][128 B]) | q_rope [16 rows][128 B]
constexpr int kPBytes = 2048;         // P8 [64 keys][32 B: hi 16 heads | lo 16 heads], MN-major, SWIZZLE_32B
constexpr int kOffQ = 0;
constexpr int kOffKV = 2 * kQBufBytes;
constexpr int kOffRopeRing = kOffKV + kStages * kStageBytes;
constexpr int kOffP = kOffRopeRing + kRopeSlots * kSlotBytes;
constexpr int kOffSmall = kOffP + 2 * kPBytes;
constexpr int kSmallBytes = 4096;
constexpr int kSmemBytes = kOffSmall + kSmallBytes + 1024;
static_assert(kSmemBytes <= 232448, "exceeds the per-CTA shared memory limit");
static_assert(kOffKV % 1024 == 0 && kOffP % 1024 == 0, "operand tiles must stay 1024-B aligned");

constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0;    // S^T buffers at columns 0 and 96: [0,32) boxes 0-1 hi|lo, [32,64) boxes 2-3 hi|lo, [64,80) RoPE
constexpr uint32_t kSBuf = 96;
constexpr uint32_t kColO = 192;  // O^T of item parity r, block b at 192 + 128 r + 32 b: [0,16) from P hi, [16,32) from P lo
constexpr uint32_t kOBuf = 128;
// The reference m sits kHeadroom binades below the largest y seen when it was last refreshed, and is refreshed when some
// y exceeds it by more than kRefresh: P8 = 2^(y - m) <= 2^8 = 256 < 448, and a weight 2^-10 below the largest still is a
// normal e4m3 number (2^-6).
constexpr float kHeadroom = 4.0f;
constexpr float kRefresh = 8.0f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kMinusHuge = -1.0e30f;

struct Small8 {
    uint64_t q_full[2], q_empty[2], kv_full[kStages][2], kv_empty[kStages], rope_full[kRopeSlots], rope_empty[kRopeSlots], s_full[2], s_empty[2], p_full[2], pv_done[2], o_full[2], o_empty[2], stat_full[2], stat_empty[2];
    uint64_t item_full[2], item_empty[2];
    int32_t item_ring[2];
    uint32_t tmem_base;
    uint32_t pad;
    alignas(16) float ginv[2][16];             // 1 / g of the item's query rows (written with its q by the epilogue warps)
    alignas(16) float scales[kStages][kPage];  // the page's token scales (bulk-copied with its first box)
    float m_ref[16];
    float alpha[16];
    float red[4][16];
    float stat_m[2][16];  // [item parity]: the item's final reference and row sums, handed to the epilogue warps
    float stat_l[2][16];
};
static_assert(sizeof(Small8) <= kSmallBytes, "Small8 does not fit");

struct K8Params {
    const WorkItem* items;
    int32_t n_items;
    int32_t* counters;
    const int32_t* dec_pt;
    int32_t dec_stride;
    const uint8_t* pool8;
    const uint4* q;      // q_dec, bf16 [n_dec][16][576]
    // kairos_fp8_mixed_step: items with q_index >= n_dec are the chunk's tokens, each run as a one-token request over the chunk's own
    // sequence (n_keys = P + j + 1): same kernel, the chunk's page table, query and output buffers
    int32_t n_dec;
    const int32_t* chunk_pt;
    const uint4* q_chunk;
    __nv_bfloat16* out_chunk;
    float* lse_chunk;
    __nv_bfloat16* out_dec;
    float* lse_dec;
    uint8_t* partials;
    float scale_log2;
    int32_t static_first;
};

__device__ __forceinline__ WorkItem load_item8(const WorkItem* p) {
    const int4 a = __ldg(reinterpret_cast<const int4*>(p));
    const int4 b = __ldg(reinterpret_cast<const int4*>(p) + 1);
    WorkItem w;
    w.kind = a.x; w.q_index = a.y; w.page_begin = a.z; w.page_end = a.w;
    w.n_keys = b.x; w.n_q = b.y; w.partial_slot = b.z; w.cost = b.w;
    return w;
}
__device__ __forceinline__ void tma_load_3d(uint32_t smem_dst, const CUtensorMap* map, uint64_t* bar, int32_t c0, int32_t c1, int32_t c2,
                                            uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5}], [%2], %6;"
        ::"r"(smem_dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(smem_dst), "l"(reinterpret_cast<uint64_t>(gsrc)), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2(float x) {
    float y;
    asm("lg2.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
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
__device__ __forceinline__ void st_f32_evict_last(float* p, float v) {
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(kEvictLast) : "memory");
}

// softmax / correction / epilogue of one decode split.  Warp sw: TMEM lane quadrant (sw + 2) & 3 (16 of its lanes hold the
// M=64 accumulator rows = keys), heads 8 (sw >> 2) .. + 8.
__device__ __forceinline__ void softmax_item8(Small8* sm, uint8_t* kv, uint8_t* pbuf, const WorkItem& w, const K8Params& p, uint32_t tmem,
                                              int sw, int lane, uint32_t& g, uint32_t it) {
    constexpr int NC = 8;
    const int w4 = (sw + 2) & 3;
    const int cbase = (sw >> 2) * NC;
    const int tid_s = sw * 32 + lane;
    const bool lane_ok = lane < 16;
    const int tok_in_page = w4 * 16 + lane;
    const int ip = it & 1;  // O^T accumulator and statistics rows of this item
    float l[NC], gi[NC];
    mbar_wait(&sm->q_full[ip], (it >> 1) & 1);  // the gains are written with the item's q
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        l[c] = 0.f;
        gi[c] = sm->ginv[ip][cbase + c] * p.scale_log2;  // 1/g_h folded with sigma * log2(e)
    }
    if (tid_s < 16) sm->m_ref[tid_s] = kMinusHuge;
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->q_empty[ip]);  // with the S warps' commits: the q buffer (and its gains) may be refilled
    named_sync(1);

    const int npages = w.page_end - w.page_begin;
    for (int pg = 0; pg < npages; ++pg, ++g) {
        const int b = g & 1;
        const int st = g % kStages;
        // the token scales came with the page's first boxes, long before its S product completes: fetch them first
        mbar_wait(&sm->kv_full[st][0], (g / kStages) & 1);
        const float sc = lane_ok ? sm->scales[st][tok_in_page] : 1.f;
        const int page = w.page_begin + pg;
        const int key_pos = page * kPage + tok_in_page;
        const bool ok = lane_ok && key_pos < w.n_keys;
        const float lsc = lg2(sc), rs = ok ? __fdividef(1.f, sc) : 0.f;

        mbar_wait(&sm->s_full[b], (g >> 1) & 1);
        tc_fence_after();
        float xa[2][NC], xb[2][NC], xr[NC];
        const uint32_t sbase = tmem_addr(tmem, w4 * 32, kColS + b * kSBuf + cbase);
        tmem_ld8(sbase, *reinterpret_cast<uint32_t(*)[8]>(xa[0]));
        tmem_ld8(sbase + 16, *reinterpret_cast<uint32_t(*)[8]>(xa[1]));
        tmem_ld8(sbase + 32, *reinterpret_cast<uint32_t(*)[8]>(xb[0]));
        tmem_ld8(sbase + 48, *reinterpret_cast<uint32_t(*)[8]>(xb[1]));
        tmem_ld8(sbase + 64, *reinterpret_cast<uint32_t(*)[8]>(xr));
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->s_empty[b]);
        float y[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float s8 = (xa[0][c] + xa[1][c]) + (xb[0][c] + xb[1][c]);  // fixed order: the result never depends on timing
            const float v = fmaf(s8 * sc, gi[c], xr[c] * p.scale_log2) + lsc;
            y[c] = ok ? v : -INFINITY;
        }
        float dmax = -INFINITY;
#pragma unroll
        for (int c = 0; c < NC; ++c) dmax = fmaxf(dmax, y[c] - sm->m_ref[cbase + c]);
        const bool need = named_or(2, dmax > kRefresh);
        if (need) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                const float wm = warp_max(y[c]);
                if (lane == c) sm->red[w4][cbase + c] = wm;
            }
            named_sync(1);
            if (tid_s < 16) {
                const float tm = fmaxf(fmaxf(sm->red[0][tid_s], sm->red[1][tid_s]), fmaxf(sm->red[2][tid_s], sm->red[3][tid_s]));
                const float mo = sm->m_ref[tid_s];
                const float mn = fmaxf(mo, tm - kHeadroom);
                sm->m_ref[tid_s] = mn;
                sm->alpha[tid_s] = ex2(mo - mn);
            }
            named_sync(1);
            if (pg > 0) {  // O^T and l are relative to the old reference: rescale (rare)
                mbar_wait(&sm->pv_done[(g - 1) & 1], ((g - 1) >> 1) & 1);
                tc_fence_after();
#pragma unroll
                for (int b4 = 0; b4 < 4; ++b4)
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
                        uint32_t r[NC];
                        const uint32_t ta = tmem_addr(tmem, w4 * 32, kColO + ip * kOBuf + b4 * 32 + half * 16 + cbase);
                        tmem_ld8(ta, *reinterpret_cast<uint32_t(*)[8]>(r));
                        tmem_wait_ld();
#pragma unroll
                        for (int i = 0; i < NC; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * sm->alpha[cbase + i]);
                        tmem_st8(ta, *reinterpret_cast<const uint32_t(*)[8]>(r));
                    }
                tmem_wait_st();
#pragma unroll
                for (int c = 0; c < NC; ++c) l[c] *= sm->alpha[cbase + c];
            }
        }
        uint32_t chi[NC / 2], clo[NC / 2];
#pragma unroll
        for (int c = 0; c < NC; c += 2) {
            const float p0 = ex2(y[c] - sm->m_ref[cbase + c]), p1 = ex2(y[c + 1] - sm->m_ref[cbase + c + 1]);
            l[c] = fmaf(p0, rs, l[c]);
            l[c + 1] = fmaf(p1, rs, l[c + 1]);
            chi[c / 2] = e4m3x2(p0, p1);
            const float2 hv = e4m3x2_value(chi[c / 2]);
            clo[c / 2] = e4m3x2(p0 - hv.x, p1 - hv.y);
        }
        if (lane_ok && (page + 1) * kPage > w.n_keys && key_pos >= w.n_keys) {
            // a stale slot of the sequence's last page: its P8 column is 0, but the PV MMA still multiplies the page's codes and
            // 0 * NaN = NaN.  Zero the token's 128 B in two of the four latent boxes (the other column half takes the rest).
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                uint4* dst = reinterpret_cast<uint4*>(kv + st * kStageBytes + ((sw >> 2) * 2 + c) * kSlotBytes + tok_in_page * 128);
#pragma unroll
                for (int j = 0; j < 8; ++j) dst[j] = make_uint4(0u, 0u, 0u, 0u);
            }
        }
        if (g >= 2) mbar_wait(&sm->pv_done[b], ((g - 2) >> 1) & 1);  // PV of page g - 2 has read this P buffer
        if (lane_ok) {
            uint8_t* pb = pbuf + b * kPBytes;
            const uint32_t kk = uint32_t(tok_in_page);
            // P8 is the MN-major B operand [64 keys][32 B: hi terms of heads 0-15 | lo terms], SWIZZLE_32B (the 16-byte chunk index
            // is XORed with bit 2 of the row): this thread's key row takes two 8-byte stores (sixteen byte stores into a K-major
            // tile cost 144 bank conflicts per page and 4 us of the step)
            const uint32_t sx = (kk >> 2) & 1u;
            *reinterpret_cast<uint2*>(pb + kk * 32u + ((0u ^ sx) << 4) + uint32_t(cbase)) = make_uint2(chi[0] | (chi[1] << 16), chi[2] | (chi[3] << 16));
            *reinterpret_cast<uint2*>(pb + kk * 32u + ((1u ^ sx) << 4) + uint32_t(cbase)) = make_uint2(clo[0] | (clo[1] << 16), clo[2] | (clo[3] << 16));
        }
        fence_proxy_async_smem();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm->p_full[b]);
    }
    // ---- hand the row statistics to the epilogue warps (they drain this item's O^T while these warps start the next item)
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        float v = l[c];
        v += __shfl_xor_sync(0xffffffffu, v, 8);
        v += __shfl_xor_sync(0xffffffffu, v, 4);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        v += __shfl_xor_sync(0xffffffffu, v, 1);  // lanes 0..15 hold the data, lanes 16..31 zeros
        if (lane == c) sm->red[w4][cbase + c] = v;
    }
    named_sync(1);
    if (tid_s < 16) {
        mbar_wait(&sm->stat_empty[ip], ((it >> 1) & 1) ^ 1);  // the epilogue of item it - 2 has read this pair of rows
        sm->stat_l[ip][tid_s] = sm->red[0][tid_s] + sm->red[1][tid_s] + sm->red[2][tid_s] + sm->red[3][tid_s];
        sm->stat_m[ip][tid_s] = sm->m_ref[tid_s];
    }
    named_sync(2);  // m_ref / red are free for the next item; the statistics are written
    if (tid_s == 0) mbar_arrive(&sm->stat_full[ip]);
}

// Query preparation of one item by the four epilogue warps (warp r: heads 4r .. 4r + 3).  Row (item, h) of the latent part is scaled
// by the power of two g that puts its largest magnitude in [128, 256) and split into two e4m3 numbers, hi = rne(q g) and
// lo = rne(q g - hi), written straight into the B-operand tiles of the S MMAs: four [32 rows][128 B] SWIZZLE_128B boxes (rows 0-15
// the hi terms of heads 0-15, rows 16-31 the lo terms), the bf16 RoPE part as a [16 rows][128 B] box, and 1 / g per head.
__device__ __forceinline__ void prepare_q8(Small8* sm, uint8_t* qdst, int qb, const uint4* rows, int r, int lane) {
    constexpr int kRowVecs = kTokenBytes / 16;  // 72
    {   // RoPE part: 8 x 16 B per head, this warp's four heads in one pass
        const int h = 4 * r + (lane >> 3), c = lane & 7;
        *reinterpret_cast<uint4*>(qdst + kQ8Bytes + sw128_offset(uint32_t(h), uint32_t(c))) = __ldg(rows + h * kRowVecs + 64 + c);
    }
    uint4 ra[4], rb[4];  // lane L owns elements [16 L, 16 L + 16) of a row; the four rows are in flight together
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        ra[u] = __ldg(rows + (4 * r + u) * kRowVecs + lane * 2);
        rb[u] = __ldg(rows + (4 * r + u) * kRowVecs + lane * 2 + 1);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int h = 4 * r + u;
        const uint32_t wv[8] = {ra[u].x, ra[u].y, ra[u].z, ra[u].w, rb[u].x, rb[u].y, rb[u].z, rb[u].w};
        float v[16];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            v[2 * k] = bf16_lo(wv[k]);
            v[2 * k + 1] = bf16_hi(wv[k]);
        }
        float amax = 0.f;
#pragma unroll
        for (int k = 0; k < 16; ++k) amax = fmaxf(amax, fabsf(v[k]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        int ex = 8;
        if (amax > 0.f) (void)frexpf(amax, &ex);  // amax = f * 2^ex, f in [0.5, 1)
        const int ge = min(8 - ex, 100);          // gain exponent: amax * 2^ge in [128, 256) (capped for denormal-small rows)
        const float gn = ldexpf(1.f, ge);
        uint32_t chi[4], clo[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t ch[2], cl[2];
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const float x0 = v[4 * k + 2 * t] * gn, x1 = v[4 * k + 2 * t + 1] * gn;
                ch[t] = e4m3x2(x0, x1);
                const float2 hv = e4m3x2_value(ch[t]);
                cl[t] = e4m3x2(x0 - hv.x, x1 - hv.y);
            }
            chi[k] = ch[0] | (ch[1] << 16);
            clo[k] = cl[0] | (cl[1] << 16);
        }
        uint8_t* box = qdst + (lane >> 3) * 4096;
        *reinterpret_cast<uint4*>(box + sw128_offset(uint32_t(h), uint32_t(lane & 7))) = make_uint4(chi[0], chi[1], chi[2], chi[3]);
        *reinterpret_cast<uint4*>(box + sw128_offset(uint32_t(16 + h), uint32_t(lane & 7))) = make_uint4(clo[0], clo[1], clo[2], clo[3]);
        if (lane == 0) sm->ginv[qb][h] = ldexpf(1.f, -ge);
    }
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->q_full[qb]);
}

// Epilogue of one decode split (warps 12-15, one per TMEM lane quadrant): O^T of the item's accumulator -> bf16 output rows, or the
// unnormalised fp32 partial of a KV split.  Runs beside the next item's pages (O^T is double-buffered by item parity).
__device__ __forceinline__ void epilogue_item8(Small8* sm, const WorkItem& w, const K8Params& p, uint32_t tmem, int w4, int lane, uint32_t it) {
    const int ip = it & 1;
    mbar_wait(&sm->stat_full[ip], (it >> 1) & 1);
    const bool is_final = w.partial_slot < 0;
    float linv[kHeads];
    {
        const int h = lane & 15;
        const float L = sm->stat_l[ip][h], m = sm->stat_m[ip][h];
        const float mli = __fdividef(1.f, L);
        if (w4 == 0 && lane < kHeads) {
            if (is_final) {
                float* lse = w.q_index < p.n_dec ? p.lse_dec : p.lse_chunk;
                const int row = w.q_index < p.n_dec ? w.q_index : w.q_index - p.n_dec;
                if (lse) lse[size_t(row) * kHeads + h] = (m + lg2(L)) * kLn2;
            } else {
                float* ml = reinterpret_cast<float*>(p.partials + size_t(w.partial_slot) * kPartialSlotBytes + size_t(kHeads) * kLatent * 4);
                ml[h] = m;
                ml[kHeads + h] = L;
            }
        }
#pragma unroll
        for (int c = 0; c < kHeads; ++c) linv[c] = __shfl_sync(0xffffffffu, mli, c);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->stat_empty[ip]);
    mbar_wait(&sm->o_full[ip], (it >> 1) & 1);  // all PV MMAs of the item are complete
    tc_fence_after();
    // O^T block b4: lane = latent dim 128 b4 + 32 w4 + lane; columns [0,16) from P hi, [16,32) from P lo.  The loads of block
    // b4 + 1 are in flight while block b4 is converted and stored.
    uint32_t rr[2][2 * kHeads];
    auto load_block = [&](int b4, uint32_t* r) {
        tmem_ld16(tmem_addr(tmem, w4 * 32, kColO + ip * kOBuf + b4 * 32), *reinterpret_cast<uint32_t(*)[16]>(r));
        tmem_ld16(tmem_addr(tmem, w4 * 32, kColO + ip * kOBuf + b4 * 32 + 16), *reinterpret_cast<uint32_t(*)[16]>(r + kHeads));
    };
    load_block(0, rr[0]);
#pragma unroll
    for (int b4 = 0; b4 < 4; ++b4) {
        tmem_wait_ld();
        if (b4 < 3) load_block(b4 + 1, rr[(b4 + 1) & 1]);
        const uint32_t* r = rr[b4 & 1];
        const int d = b4 * 128 + w4 * 32 + lane;
        if (is_final) {
            __nv_bfloat16* o = (w.q_index < p.n_dec ? p.out_dec + size_t(w.q_index) * kHeads * kLatent
                                                    : p.out_chunk + size_t(w.q_index - p.n_dec) * kHeads * kLatent) + d;
#pragma unroll
            for (int i = 0; i < kHeads; ++i) o[i * kLatent] = __float2bfloat16_rn((__uint_as_float(r[i]) + __uint_as_float(r[kHeads + i])) * linv[i]);
        } else {
            float* o = reinterpret_cast<float*>(p.partials + size_t(w.partial_slot) * kPartialSlotBytes) + d;
#pragma unroll
            for (int i = 0; i < kHeads; ++i) st_f32_evict_last(o + i * kLatent, __uint_as_float(r[i]) + __uint_as_float(r[kHeads + i]));
        }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(&sm->o_empty[ip]);
}

// S MMAs of one decode split, in two halves issued by two warps: half 0 = latent boxes 0-1 into columns [0,32) of the S buffer,
// half 1 = latent boxes 2-3 into [32,64) and the RoPE box into [64,80).  Each half accumulates in a fixed order.
template <int HALF>
__device__ __forceinline__ void s_item8(Small8* sm, uint32_t tmem, uint32_t q_base, uint32_t kv_base, int npages, uint32_t g0, uint32_t qbuf,
                                        uint32_t qfull_parity) {
    constexpr uint32_t idesc_s8 = make_idesc_e4m3(64, 32, 0, 0);  // S8^T = K8 [Qhi;Qlo]^T: A K-major, B K-major
    constexpr uint32_t idesc_sr = make_idesc_bf16(64, 16, 0, 0);  // SR^T = KR QR^T
    constexpr uint32_t desc_hi = smem_desc_hi(1024);
    mbar_wait(&sm->q_full[qbuf], qfull_parity);
    for (int s = 0; s < npages; ++s) {
        const uint32_t gg = g0 + s;
        const uint32_t sb = gg & 1, st = gg % kStages, par = (gg / kStages) & 1;
        mbar_wait(&sm->s_empty[sb], ((gg >> 1) & 1) ^ 1);
        mbar_wait(&sm->kv_full[st][HALF], par);
        tc_fence_after();
#pragma unroll
        for (uint32_t bb = 0; bb < 2; ++bb) {
            const uint32_t b = 2 * HALF + bb;
            const uint32_t ka_lo = smem_desc_lo(kv_base + st * kStageBytes + b * kSlotBytes, 16);
            const uint32_t qb_lo = smem_desc_lo(q_base + b * 4096, 16);
#pragma unroll
            for (uint32_t j = 0; j < 4; ++j)
                umma_f8_ss_lohi(tmem + kColS + sb * kSBuf + 32 * HALF, ka_lo + ((j * 32) >> 4), desc_hi, qb_lo + ((j * 32) >> 4), desc_hi,
                                idesc_s8, !(bb == 0 && j == 0));
        }
        if (HALF == 1) {
            mbar_wait(&sm->rope_full[gg & 1], (gg >> 1) & 1);
            tc_fence_after();
            const uint32_t ka_lo = smem_desc_lo(kv_base + kStages * kStageBytes + (gg & 1) * kSlotBytes, 16);
            const uint32_t qb_lo = smem_desc_lo(q_base + kQ8Bytes, 16);
#pragma unroll
            for (uint32_t j = 0; j < 4; ++j)
                umma_bf16_ss_lohi(tmem + kColS + sb * kSBuf + 64, ka_lo + ((j * 32) >> 4), desc_hi, qb_lo + ((j * 32) >> 4), desc_hi, idesc_sr, j > 0);
        }
        umma_commit_elect(&sm->s_full[sb]);
        if (HALF == 1) umma_commit_elect(&sm->rope_empty[gg & 1]);  // the RoPE box is only ever read by these MMAs
        if (s == npages - 1) umma_commit_elect(&sm->q_empty[qbuf]);
    }
}

// PV MMAs (warp kPvWarp): O^T block b4 += V8^T block b4 [128 dims x 64 keys] (MN-major view of latent box b4) . P8^T
__device__ __forceinline__ void pv_item8(Small8* sm, uint32_t tmem, uint32_t kv_base, uint32_t p_base, int npages, uint32_t g0, uint32_t it) {
    constexpr uint32_t idesc_o8 = make_idesc_e4m3(128, 32, 1, 1);
    constexpr uint32_t pdesc_hi = smem_desc_hi_sw32(256);  // P8: 8 key rows of 32 B per swizzle atom
    constexpr uint32_t desc_hi = smem_desc_hi(1024);
    for (int pv = 0; pv < npages; ++pv) {
        const uint32_t gg = g0 + pv;
        const uint32_t pst = gg & 1, pph = (gg >> 1) & 1, st = gg % kStages;
        mbar_wait(&sm->p_full[pst], pph);
        if (pv == 0) mbar_wait(&sm->o_empty[it & 1], ((it >> 1) & 1) ^ 1);  // the epilogue of item it - 2 has drained this accumulator
        tc_fence_after();
        const uint32_t pb_lo = smem_desc_lo(p_base + pst * kPBytes, 16);
#pragma unroll
        for (uint32_t b4 = 0; b4 < 4; ++b4) {
            const uint32_t va_lo = smem_desc_lo(kv_base + st * kStageBytes + b4 * kSlotBytes, 8192);
#pragma unroll
            for (uint32_t ks = 0; ks < 2; ++ks)  // 32 keys per instruction: 32 rows of 128 B further down the box
                umma_f8_ss_lohi(tmem + kColO + (it & 1) * kOBuf + b4 * 32, va_lo + ((ks * 4096) >> 4), desc_hi, pb_lo + ((ks * 1024) >> 4), pdesc_hi, idesc_o8,
                                (pv > 0 || ks > 0));
        }
        umma_commit_elect(&sm->kv_empty[st]);  // the whole stage (the S MMAs of this page completed before its softmax started)
        umma_commit_elect(&sm->pv_done[pst]);
        if (pv == npages - 1) umma_commit_elect(&sm->o_full[it & 1]);
    }
}

__global__ void __launch_bounds__(kThreads, 1)
kairos_fp8_decode_kernel(const __grid_constant__ CUtensorMap lat_map, const __grid_constant__ CUtensorMap rope_map,
                         const K8Params p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    Small8* sm = reinterpret_cast<Small8*>(base + kOffSmall);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < 2; ++i) {
            mbar_init(&sm->q_full[i], 4);
            mbar_init(&sm->q_empty[i], 2 + kSoftmaxWarps);
            mbar_init(&sm->s_full[i], 2);
            mbar_init(&sm->s_empty[i], kSoftmaxWarps);
            mbar_init(&sm->item_full[i], 1);
            mbar_init(&sm->item_empty[i], 3 + kSoftmaxWarps + 4);
            mbar_init(&sm->p_full[i], kSoftmaxWarps);
            mbar_init(&sm->pv_done[i], 1);
        }
        for (int i = 0; i < kStages; ++i) {
            mbar_init(&sm->kv_full[i][0], 1);
            mbar_init(&sm->kv_full[i][1], 1);
            mbar_init(&sm->kv_empty[i], 1);
        }
        for (int i = 0; i < kRopeSlots; ++i) {
            mbar_init(&sm->rope_full[i], 1);
            mbar_init(&sm->rope_empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&sm->o_full[i], 1);
            mbar_init(&sm->o_empty[i], 4);
            mbar_init(&sm->stat_full[i], 1);
            mbar_init(&sm->stat_empty[i], 4);
        }
        fence_barrier_init();
    }
    if (warp == 0 && lane == 0) {
        prefetch_tensormap(&lat_map);
        prefetch_tensormap(&rope_map);
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the combine grid may pre-launch
    if (warp == 1) tmem_alloc(&sm->tmem_base, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm->tmem_base;

    if (warp == 0) {
        // ================= producer =================
        uint32_t g = 0;
        const uint32_t kv_u32 = smem_u32(base + kOffKV);
        for (uint32_t it = 0;; ++it) {
            int idx = int(blockIdx.x);
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
            const WorkItem w = load_item8(p.items + idx);
            const int npages = w.page_end - w.page_begin;
            const bool is_chunk = w.q_index >= p.n_dec;
            const int32_t* pt = (is_chunk ? p.chunk_pt : p.dec_pt + size_t(w.q_index) * p.dec_stride) + w.page_begin;
            const uint64_t policy = is_chunk ? kEvictLast : kEvictFirst;  // the chunk's pages are re-read by every later token of the chunk
            for (int i = 0; i < npages; i += 32) {
                const int my = (i + lane < npages) ? __ldg(pt + i + lane) : 0;
                const int cnt = min(32, npages - i);
                for (int j = 0; j < cnt; ++j, ++g) {
                    const int pid = __shfl_sync(0xffffffffu, my, j);
                    if (lane == 0) {
                        const uint32_t st = g % kStages, par = ((g / kStages) & 1) ^ 1;
                        mbar_wait(&sm->kv_empty[st], par);
                        mbar_arrive_expect_tx(&sm->kv_full[st][0], 2 * kSlotBytes + kPage * 4);
                        mbar_arrive_expect_tx(&sm->kv_full[st][1], 2 * kSlotBytes);
#pragma unroll
                        for (int b = 0; b < 4; ++b)
                            tma_load_3d(kv_u32 + st * kStageBytes + b * kSlotBytes, &lat_map, &sm->kv_full[st][b >> 1], b * 128, 0, pid, policy);
                        mbar_wait(&sm->rope_empty[g & 1], ((g >> 1) & 1) ^ 1);  // S of page g - 2 retired long before a latent stage frees
                        mbar_arrive_expect_tx(&sm->rope_full[g & 1], kSlotBytes);
                        tma_load_3d(kv_u32 + kStages * kStageBytes + (g & 1) * kSlotBytes, &rope_map, &sm->rope_full[g & 1], 0, 0, pid, policy);
                        bulk_load(smem_u32(sm->scales[st]), p.pool8 + size_t(pid) * kPage8Bytes + kOffScale8, kPage * 4, &sm->kv_full[st][0],
                                  policy);
                    }
                }
            }
        }
    } else if (warp == 1 || warp == kPvWarp || warp == kSbWarp) {
        // ================= MMA issuers =================
        const uint32_t q_base = smem_u32(base + kOffQ), kv_base = smem_u32(base + kOffKV), p_base = smem_u32(base + kOffP);
        uint32_t g = 0;
        for (uint32_t it = 0;; ++it) {
            mbar_wait(&sm->item_full[it & 1], (it >> 1) & 1);
            const int idx = __shfl_sync(0xffffffffu, sm->item_ring[it & 1], 0);
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->item_empty[it & 1]);
            __syncwarp();
            if (idx < 0) break;
            const WorkItem w = load_item8(p.items + idx);
            const int npages = __shfl_sync(0xffffffffu, w.page_end - w.page_begin, 0);
            if (warp == 1) s_item8<0>(sm, tmem, q_base + (it & 1u) * kQBufBytes, kv_base, npages, g, it & 1u, (it >> 1) & 1u);
            else if (warp == kSbWarp) s_item8<1>(sm, tmem, q_base + (it & 1u) * kQBufBytes, kv_base, npages, g, it & 1u, (it >> 1) & 1u);
            else pv_item8(sm, tmem, kv_base, p_base, npages, g, it);
            g += npages;
        }
    } else if (warp >= kEpiWarp) {
        // ================= epilogue warps =================
        // Per item: first its query rows (the S warps need them as soon as the item's first page has landed; the producer publishes an
        // item about five pages ahead of that), then the output of the PREVIOUS item, whose last PV retires about now.
        WorkItem prev{};
        for (uint32_t it = 0;; ++it) {
            mbar_wait(&sm->item_full[it & 1], (it >> 1) & 1);
            const int idx = sm->item_ring[it & 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->item_empty[it & 1]);
            WorkItem w{};
            if (idx >= 0) {
                w = load_item8(p.items + idx);
                const int qb = int(it & 1);
                mbar_wait(&sm->q_empty[qb], ((it >> 1) & 1) ^ 1);
                const uint4* qrows = w.q_index < p.n_dec ? p.q + size_t(w.q_index) * kHeads * (kTokenBytes / 16)
                                                         : p.q_chunk + size_t(w.q_index - p.n_dec) * kHeads * (kTokenBytes / 16);
                prepare_q8(sm, base + kOffQ + qb * kQBufBytes, qb, qrows, warp - kEpiWarp, lane);
            }
            if (it > 0) epilogue_item8(sm, prev, p, tmem, warp & 3, lane, it - 1);
            if (idx < 0) break;
            prev = w;
        }
    } else {
        // ================= softmax / correction warps =================
        const int sw = warp - 2;
        uint32_t g = 0;
        for (uint32_t it = 0;; ++it) {
            mbar_wait(&sm->item_full[it & 1], (it >> 1) & 1);
            const int idx = sm->item_ring[it & 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->item_empty[it & 1]);
            if (idx < 0) break;
            const WorkItem w = load_item8(p.items + idx);
            softmax_item8(sm, base + kOffKV, base + kOffP, w, p, tmem, sw, lane, g, it);
        }
    }

    tc_fence_before();
    __syncthreads();
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

}  // namespace

int fp8_attach(kairos_ctx* ctx, void* pool8, int32_t num_pages) {
    Fp8State& f = ctx->fp8;
    f.attached = false;
    {   // latent codes: [page][64 tokens][512 B], boxes of 128 codes x 64 tokens
        const uint64_t dims[3] = {uint64_t(kLatent), uint64_t(kPage), uint64_t(num_pages)};
        const uint64_t strides[2] = {uint64_t(kLatent), uint64_t(kPage8Bytes)};
        const uint32_t box[3] = {128, uint32_t(kPage), 1};
        if (int rc = encode_tiled_map(&f.lat_map, /*u8=*/true, 3, pool8, dims, strides, box)) return rc;
    }
    {   // RoPE keys: bf16 [page][64 tokens][64] behind the codes of each page
        const uint64_t dims[3] = {uint64_t(kRope), uint64_t(kPage), uint64_t(num_pages)};
        const uint64_t strides[2] = {uint64_t(kRope * 2), uint64_t(kPage8Bytes)};
        const uint32_t box[3] = {uint32_t(kRope), uint32_t(kPage), 1};
        if (int rc = encode_tiled_map(&f.rope_map, /*u8=*/false, 3, static_cast<uint8_t*>(pool8) + kOffRope8, dims, strides, box)) return rc;
    }
    KAIROS_CUDA_TRY(cudaFuncSetAttribute(kairos_fp8_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    f.pool8 = pool8;
    f.num_pages = num_pages;
    f.attached = true;
    return KAIROS_OK;
}

int launch_fp8_append(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens, const int32_t* page_table,
                      int32_t start_pos, cudaStream_t stream) {
    fp8_append_kernel<<<(n_tokens + 7) / 8, 256, 0, stream>>>(static_cast<uint8_t*>(ctx->fp8.pool8), reinterpret_cast<const uint4*>(latent),
                                                              reinterpret_cast<const uint4*>(k_rope), page_table, n_tokens, start_pos, nullptr, 0);
    KAIROS_CUDA_TRY(cudaGetLastError());
    return KAIROS_OK;
}

int launch_fp8_append_decode(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n, const int32_t* page_tables,
                             int32_t table_stride, const int32_t* positions, cudaStream_t stream) {
    fp8_append_kernel<<<(n + 7) / 8, 256, 0, stream>>>(static_cast<uint8_t*>(ctx->fp8.pool8), reinterpret_cast<const uint4*>(latent),
                                                       reinterpret_cast<const uint4*>(k_rope), page_tables, n, 0, positions, table_stride);
    KAIROS_CUDA_TRY(cudaGetLastError());
    return KAIROS_OK;
}

int launch_fp8_decode(kairos_ctx* ctx, const StepArgs& a, const WorkItem* dev_items, int32_t n_items, cudaStream_t stream) {
    Fp8State& f = ctx->fp8;
    K8Params p;
    p.items = dev_items;
    p.n_items = n_items;
    p.counters = reinterpret_cast<int32_t*>(ctx->cfg.workspace);
    p.dec_pt = a.dec_page_tables;
    p.dec_stride = a.dec_table_stride;
    p.pool8 = static_cast<const uint8_t*>(f.pool8);
    p.q = reinterpret_cast<const uint4*>(a.q_dec);
    p.n_dec = a.n_dec;
    p.chunk_pt = a.chunk_page_table;
    p.q_chunk = reinterpret_cast<const uint4*>(a.q_chunk);
    p.out_chunk = reinterpret_cast<__nv_bfloat16*>(a.out_chunk);
    p.lse_chunk = a.lse_chunk;
    p.out_dec = reinterpret_cast<__nv_bfloat16*>(a.out_dec);
    p.lse_dec = a.lse_dec;
    p.partials = reinterpret_cast<uint8_t*>(ctx->cfg.workspace) + 256;
    p.scale_log2 = ctx->cfg.softmax_scale * 1.4426950408889634f;
    p.static_first = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(std::max(1, std::min(n_items, umma_resident_ctas(ctx)))), 1, 1);
    cfg.blockDim = dim3(kThreads, 1, 1);
    cfg.dynamicSmemBytes = kSmemBytes;
    cfg.stream = stream;
    cfg.attrs = nullptr;
    cfg.numAttrs = 0;
    KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, kairos_fp8_decode_kernel, f.lat_map, f.rope_map, p));
    return KAIROS_OK;
}

}  // namespace kairos
