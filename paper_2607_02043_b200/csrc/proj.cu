// the projections either side of the attention (the model is DeepSeek-V2-Lite; absorbed
// MLA as restated in SURVEY.md 8(c)): the query "absorption" q_lat[n,h,:] = q_nope[n,h,:] . W_UK[h] (128 -> 512) that
// produces the latent part of the q rows kairos_mixed_step takes, and the value up-projection v[n,h,:] = o_lat[n,h,:] . W_UV[h]
// (512 -> 128) that consumes its outputs.  Both are per-head GEMMs with a 128-token M tile on tcgen05: operands K-major in
// shared memory through TMA (SWIZZLE_128B), fp32 accumulator in tensor memory, bf16 RNE stores.
#include <cuda_bf16.h>

#include "kairos_internal.h"
#include "umma_ptx.cuh"

namespace kairos {
namespace {
using namespace ptx;

constexpr int kProjThreads = 192;  // warp 0 TMA producer, warp 1 MMA issuer + TMEM owner, warps 2-5 epilogue (one TMEM lane quadrant each)
constexpr int kProjTile = 128;     // tokens per CTA

template <int N>
struct ProjGeo {
    static constexpr int kStages = N >= 512 ? 2 : 4;
    static constexpr int kABytes = kProjTile * 128;  // [128 tokens][64 k] bf16
    static constexpr int kBBytes = N * 128;          // [N][64 k] bf16
    static constexpr int kStageBytes = kABytes + kBBytes;
    static constexpr int kSmem = kStages * kStageBytes + 256 + 1024;
    static constexpr int kNBlock = N >= 256 ? 256 : N;  // columns per MMA (and rows per TMA box of B)
};

struct ProjParams {
    __nv_bfloat16* out;      // [n][16][out_stride]
    int32_t out_stride;      // elements between heads of the output (576 for q rows, 128 for v)
    const uint4* rope_in;    // absorb: q_rope [n][16][64] copied behind the 512 latent columns; else NULL
    int32_t n;
};

template <int N, int KDIM>
__global__ void __launch_bounds__(kProjThreads, 1)
kairos_proj_kernel(const __grid_constant__ CUtensorMap a_map, const __grid_constant__ CUtensorMap b_map, const ProjParams p) {
    using G = ProjGeo<N>;
    constexpr int S = G::kStages, NB = G::kNBlock, KC = KDIM / 64;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full = reinterpret_cast<uint64_t*>(base + S * G::kStageBytes);
    uint64_t* empty = full + S;
    uint64_t* d_full = empty + S;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_full + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m0 = blockIdx.x * kProjTile, h = blockIdx.y;
    if (threadIdx.x == 0) {
        for (int i = 0; i < S; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], 1);
        }
        mbar_init(d_full, 1);
        fence_barrier_init();
        prefetch_tensormap(&a_map);
        prefetch_tensormap(&b_map);
    }
    if (warp == 1) tmem_alloc(tmem_slot, N);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {
            for (int kc = 0; kc < KC; ++kc) {
                const int st = kc % S;
                mbar_wait(&empty[st], ((kc / S) & 1) ^ 1);
                mbar_arrive_expect_tx(&full[st], G::kStageBytes);
                uint8_t* sa = base + st * G::kStageBytes;
                tma_load_2d(sa, &a_map, &full[st], h * KDIM + kc * 64, m0, kEvictFirst);  // rows past n are zero-filled
                for (int nb = 0; nb < N / NB; ++nb)
                    tma_load_2d(sa + G::kABytes + nb * NB * 128, &b_map, &full[st], kc * 64, h * N + nb * NB, kEvictLast);
            }
        }
    } else if (warp == 1) {
        constexpr uint32_t idesc = make_idesc_bf16(128, NB, 0, 0);
        constexpr uint32_t hi = smem_desc_hi(1024);
        for (int kc = 0; kc < KC; ++kc) {
            const int st = kc % S;
            mbar_wait(&full[st], (kc / S) & 1);
            tc_fence_after();
            const uint32_t a_lo = smem_desc_lo(smem_u32(base + st * G::kStageBytes), 16);
#pragma unroll
            for (int nb = 0; nb < N / NB; ++nb) {
                const uint32_t b_lo = smem_desc_lo(smem_u32(base + st * G::kStageBytes + G::kABytes + nb * NB * 128), 16);
#pragma unroll
                for (uint32_t j = 0; j < 4; ++j)
                    umma_bf16_ss_lohi(tmem + nb * NB, a_lo + ((j * 32) >> 4), hi, b_lo + ((j * 32) >> 4), hi, idesc, (kc | int(j)) != 0);
            }
            umma_commit_elect(&empty[st]);
        }
        umma_commit_elect(d_full);
    } else {
        const int q4 = warp & 3;  // TMEM lane quadrant this warp may touch
        const int row = q4 * 32 + lane;
        const int token = m0 + row;
        const bool live = token < p.n;
        __nv_bfloat16* orow = p.out + (size_t(token) * kHeads + h) * p.out_stride;
        if (p.rope_in && live) {  // the RoPE part of the q row passes through (already rotated upstream)
            const uint4* src = p.rope_in + (size_t(token) * kHeads + h) * 8;
            uint4* dst = reinterpret_cast<uint4*>(orow + kLatent);
#pragma unroll
            for (int j = 0; j < 8; ++j) dst[j] = __ldg(src + j);
        }
        mbar_wait(d_full, 0);
        tc_fence_after();
        const uint32_t lane_base = uint32_t(q4 * 32) << 16;
#pragma unroll 1
        for (int cb = 0; cb < N / 32; ++cb) {
            uint32_t r[32];
            tmem_ld32(tmem + lane_base + cb * 32, r);  // warp-collective: every lane takes part, dead rows do not store
            tmem_wait_ld();
            if (live) {
                uint4* dst = reinterpret_cast<uint4*>(orow + cb * 32);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint4 v;
                    uint32_t* vv = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const __nv_bfloat162 b2 = __floats2bfloat162_rn(__uint_as_float(r[8 * j + 2 * i]), __uint_as_float(r[8 * j + 2 * i + 1]));
                        vv[i] = *reinterpret_cast<const uint32_t*>(&b2);
                    }
                    dst[j] = v;
                }
            }
        }
        tc_fence_before();
    }
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, N);
}

template <int N, int KDIM>
int launch_proj(kairos_ctx* ctx, QMapCache* a_cache, QMapCache* b_cache, const void* a, const void* w, int32_t n, const ProjParams& p,
                cudaStream_t stream) {
    using G = ProjGeo<N>;
    // A viewed as [n rows][16*KDIM] (box 64 x 128), the weights as [16*N rows][KDIM] (box 64 x NBlock)
    if (int rc = encode_2d_map(a_cache, a, uint64_t(kHeads) * KDIM, uint64_t(n), uint64_t(kHeads) * KDIM * 2, 64, kProjTile)) return rc;
    if (int rc = encode_2d_map(b_cache, w, uint64_t(KDIM), uint64_t(kHeads) * N, uint64_t(KDIM) * 2, 64, G::kNBlock)) return rc;
    static bool attr_set = false;
    if (!attr_set) {
        KAIROS_CUDA_TRY(cudaFuncSetAttribute(kairos_proj_kernel<N, KDIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::kSmem));
        attr_set = true;
    }
    dim3 grid(unsigned((n + kProjTile - 1) / kProjTile), kHeads, 1);
    kairos_proj_kernel<N, KDIM><<<grid, kProjThreads, G::kSmem, stream>>>(a_cache->map, b_cache->map, p);
    KAIROS_CUDA_TRY(cudaGetLastError());
    (void)ctx;
    return KAIROS_OK;
}

}  // namespace

int launch_absorb_q(kairos_ctx* ctx, const void* q_nope, const void* q_rope, const void* w_uk_t, int32_t n, void* q_out, cudaStream_t stream) {
    ProjParams p{reinterpret_cast<__nv_bfloat16*>(q_out), kDim, reinterpret_cast<const uint4*>(q_rope), n};
    return launch_proj<kLatent, 128>(ctx, &ctx->proj_a[0], &ctx->proj_b[0], q_nope, w_uk_t, n, p, stream);
}

int launch_project_out(kairos_ctx* ctx, const void* o_lat, const void* w_uv_t, int32_t n, void* v_out, cudaStream_t stream) {
    ProjParams p{reinterpret_cast<__nv_bfloat16*>(v_out), 128, nullptr, n};
    return launch_proj<128, kLatent>(ctx, &ctx->proj_a[1], &ctx->proj_b[1], o_lat, w_uv_t, n, p, stream);
}

}  // namespace kairos
