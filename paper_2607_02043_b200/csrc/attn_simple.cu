// impl 0: correctness-first attention on CUDA cores -- one CTA per query token (16 heads = 16 warps), online
// softmax over 32-key tiles staged in shared memory.  Kept as a GPU-side cross-check of the tcgen05 path
// (KAIROS_IMPL=simple); it is NOT the product path and is never selected implicitly.
// Math: SURVEY.md 8(c) definition (absorbed MLA): s_t = scale*(q . [c_t|kR_t]), o = sum softmax(s)_t c_t.
#include <cuda_bf16.h>

#include "kairos_internal.h"

namespace kairos {
namespace {

constexpr int kTile = 32;                 // keys per tile (lane = key in the score phase)
constexpr int kRowStride = kDim * 2 + 16; // 1168 B: 16-B aligned, conflict-free for LDS.128 across lanes
constexpr int kThreads = kHeads * 32;     // 512
constexpr size_t kSmemBytes = size_t(kTile) * kRowStride + size_t(kHeads) * kDim * 4;  // 37,376 + 36,864

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__global__ void __launch_bounds__(kThreads, 1)
attn_simple_kernel(const uint8_t* __restrict__ pool, const __nv_bfloat16* __restrict__ q_dec,
                   const __nv_bfloat16* __restrict__ q_chunk, const int32_t* __restrict__ dec_pt, int32_t dec_stride,
                   const int32_t* __restrict__ dec_lens, const int32_t* __restrict__ chunk_pt, int32_t n_dec,
                   int32_t prefix_len, float scale, __nv_bfloat16* __restrict__ out_dec,
                   __nv_bfloat16* __restrict__ out_chunk, float* __restrict__ lse_dec, float* __restrict__ lse_chunk) {
    extern __shared__ __align__(16) uint8_t smem[];
    uint8_t* ks = smem;                                                // [32][1168 B]
    float* qs = reinterpret_cast<float*>(smem + kTile * kRowStride);   // [16][576] fp32

    const int bid = blockIdx.x;
    const __nv_bfloat16* q;
    const int32_t* pt;
    __nv_bfloat16* out;
    float* lse;
    int32_t n;
    if (bid < n_dec) {
        q = q_dec + size_t(bid) * kHeads * kDim;
        pt = dec_pt + size_t(bid) * dec_stride;
        n = dec_lens[bid];
        out = out_dec + size_t(bid) * kHeads * kLatent;
        lse = lse_dec ? lse_dec + size_t(bid) * kHeads : nullptr;
    } else {
        const int j = bid - n_dec;
        q = q_chunk + size_t(j) * kHeads * kDim;
        pt = chunk_pt;
        n = prefix_len + j + 1;
        out = out_chunk + size_t(j) * kHeads * kLatent;
        lse = lse_chunk ? lse_chunk + size_t(j) * kHeads : nullptr;
    }
    const int tid = threadIdx.x, h = tid >> 5, lane = tid & 31;
    for (int i = tid; i < kHeads * kDim; i += kThreads) qs[i] = __bfloat162float(q[i]);

    float m = -INFINITY, l = 0.f;
    float acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = 0.f;
    const float* qh = qs + h * kDim;

    for (int32_t t0 = 0; t0 < n; t0 += kTile) {
        __syncthreads();  // previous tile fully consumed (also orders the qs fill on the first pass)
        for (int i = tid; i < kTile * (kTokenBytes / 16); i += kThreads) {
            const int r = i / (kTokenBytes / 16), v = i % (kTokenBytes / 16);
            const int32_t t = t0 + r;
            uint4 val = make_uint4(0, 0, 0, 0);
            if (t < n) {
                const size_t slot = size_t(__ldg(pt + t / kPage)) * kPage + t % kPage;
                val = __ldg(reinterpret_cast<const uint4*>(pool + slot * kTokenBytes) + v);
            }
            *reinterpret_cast<uint4*>(ks + r * kRowStride + v * 16) = val;
        }
        __syncthreads();
        // scores: lane = key
        float s = 0.f;
        const uint8_t* krow = ks + lane * kRowStride;
#pragma unroll 4
        for (int v = 0; v < kTokenBytes / 16; ++v) {
            const uint4 kk = *reinterpret_cast<const uint4*>(krow + v * 16);
            const float4 qa = *reinterpret_cast<const float4*>(qh + v * 8);
            const float4 qb = *reinterpret_cast<const float4*>(qh + v * 8 + 4);
            s += qa.x * bf16_lo(kk.x) + qa.y * bf16_hi(kk.x) + qa.z * bf16_lo(kk.y) + qa.w * bf16_hi(kk.y) +
                 qb.x * bf16_lo(kk.z) + qb.y * bf16_hi(kk.z) + qb.z * bf16_lo(kk.w) + qb.w * bf16_hi(kk.w);
        }
        s = (t0 + lane < n) ? s * scale : -INFINITY;
        float tmax = s;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
        const float m_new = fmaxf(m, tmax);           // finite: key t0 is always visible
        const float corr = __expf(m - m_new);         // m = -inf on the first tile -> 0
        const float p = __expf(s - m_new);            // masked keys -> 0
        float psum = p;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) psum += __shfl_xor_sync(0xffffffffu, psum, o);
        l = l * corr + psum;
        m = m_new;
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] *= corr;
        // PV: lane owns latent dims [16*lane, 16*lane+16)
        const int kmax = min(kTile, n - t0);
        for (int k = 0; k < kmax; ++k) {
            const float pk = __shfl_sync(0xffffffffu, p, k);
            const uint4 v0 = *reinterpret_cast<const uint4*>(ks + k * kRowStride + lane * 32);
            const uint4 v1 = *reinterpret_cast<const uint4*>(ks + k * kRowStride + lane * 32 + 16);
            acc[0] += pk * bf16_lo(v0.x);  acc[1] += pk * bf16_hi(v0.x);
            acc[2] += pk * bf16_lo(v0.y);  acc[3] += pk * bf16_hi(v0.y);
            acc[4] += pk * bf16_lo(v0.z);  acc[5] += pk * bf16_hi(v0.z);
            acc[6] += pk * bf16_lo(v0.w);  acc[7] += pk * bf16_hi(v0.w);
            acc[8] += pk * bf16_lo(v1.x);  acc[9] += pk * bf16_hi(v1.x);
            acc[10] += pk * bf16_lo(v1.y); acc[11] += pk * bf16_hi(v1.y);
            acc[12] += pk * bf16_lo(v1.z); acc[13] += pk * bf16_hi(v1.z);
            acc[14] += pk * bf16_lo(v1.w); acc[15] += pk * bf16_hi(v1.w);
        }
    }
    const float inv = 1.f / l;
    __nv_bfloat16* o = out + h * kLatent + lane * 16;
    __align__(16) __nv_bfloat162 packed[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) packed[i] = __floats2bfloat162_rn(acc[2 * i] * inv, acc[2 * i + 1] * inv);
    reinterpret_cast<uint4*>(o)[0] = reinterpret_cast<uint4*>(packed)[0];
    reinterpret_cast<uint4*>(o)[1] = reinterpret_cast<uint4*>(packed)[1];
    if (lse && lane == 0) lse[h] = m + logf(l);
}

}  // namespace

int launch_attn_simple(kairos_ctx* ctx, const StepArgs& a, const int32_t* dev_lens, cudaStream_t stream) {
    static bool attr_set = false;
    if (!attr_set) {
        KAIROS_CUDA_TRY(cudaFuncSetAttribute(attn_simple_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             int(kSmemBytes)));
        attr_set = true;
    }
    const int grid = a.n_dec + a.chunk_len;
    if (grid == 0) return KAIROS_OK;
    attn_simple_kernel<<<grid, kThreads, kSmemBytes, stream>>>(
        reinterpret_cast<const uint8_t*>(ctx->cfg.pool), reinterpret_cast<const __nv_bfloat16*>(a.q_dec),
        reinterpret_cast<const __nv_bfloat16*>(a.q_chunk), a.dec_page_tables, a.dec_table_stride, dev_lens,
        a.chunk_page_table, a.n_dec, a.prefix_len, ctx->cfg.softmax_scale,
        reinterpret_cast<__nv_bfloat16*>(a.out_dec), reinterpret_cast<__nv_bfloat16*>(a.out_chunk), a.lse_dec,
        a.lse_chunk);
    KAIROS_CUDA_TRY(cudaGetLastError());
    return KAIROS_OK;
}

}  // namespace kairos
