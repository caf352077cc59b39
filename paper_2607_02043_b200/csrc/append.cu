// a1: paged latent-cache append / gather -- pure byte copies with 16-byte vector accesses.
// One cached token = 576 bf16 = 72 x 16 B (64 latent vectors + 8 RoPE-key vectors), SURVEY.md 8(a) row a1.
#include "kairos_internal.h"

namespace kairos {
namespace {

constexpr int kVecPerToken = kTokenBytes / 16;  // 72
constexpr int kLatentVecs = kLatent * 2 / 16;   // 64

// grid-stride over (token, vec); consecutive threads take consecutive 16-B vectors of one token.
__global__ void __launch_bounds__(256) append_kernel(uint4* __restrict__ pool, const uint4* __restrict__ latent,
                                                     const uint4* __restrict__ k_rope,
                                                     const int32_t* __restrict__ page_table, int32_t n_tokens,
                                                     int32_t start_pos) {
    // Launched with programmatic stream serialisation: the grid may become resident while the previous kernel of the stream
    // (typically the previous step's combine or attention kernel, which trigger launch_dependents on entry) is still
    // running, and waits here until that kernel has completed and flushed -- the launch latency is hidden, the order is not
    // relaxed (the previous step may still be reading the pages this step overwrites).
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int64_t total = int64_t(n_tokens) * kVecPerToken;
    for (int64_t i = blockIdx.x * int64_t(blockDim.x) + threadIdx.x; i < total; i += int64_t(gridDim.x) * blockDim.x) {
        const int32_t j = int32_t(i / kVecPerToken);
        const int32_t v = int32_t(i % kVecPerToken);
        const int32_t pos = start_pos + j;
        const int64_t slot = int64_t(__ldg(page_table + pos / kPage)) * kPage + pos % kPage;
        const uint4 val = v < kLatentVecs ? __ldg(latent + int64_t(j) * kLatentVecs + v)
                                          : __ldg(k_rope + int64_t(j) * (kVecPerToken - kLatentVecs) + (v - kLatentVecs));
        pool[slot * kVecPerToken + v] = val;
    }
}

// one token per request: request j writes at positions[j] through row j of page_tables.
__global__ void __launch_bounds__(256) append_decode_kernel(uint4* __restrict__ pool, const uint4* __restrict__ latent,
                                                            const uint4* __restrict__ k_rope,
                                                            const int32_t* __restrict__ page_tables,
                                                            int32_t table_stride, const int32_t* __restrict__ positions,
                                                            int32_t n) {
    const int64_t total = int64_t(n) * kVecPerToken;
    for (int64_t i = blockIdx.x * int64_t(blockDim.x) + threadIdx.x; i < total; i += int64_t(gridDim.x) * blockDim.x) {
        const int32_t j = int32_t(i / kVecPerToken);
        const int32_t v = int32_t(i % kVecPerToken);
        const int32_t pos = __ldg(positions + j);
        const int64_t slot = int64_t(__ldg(page_tables + int64_t(j) * table_stride + pos / kPage)) * kPage + pos % kPage;
        const uint4 val = v < kLatentVecs ? __ldg(latent + int64_t(j) * kLatentVecs + v)
                                          : __ldg(k_rope + int64_t(j) * (kVecPerToken - kLatentVecs) + (v - kLatentVecs));
        pool[slot * kVecPerToken + v] = val;
    }
}

__global__ void __launch_bounds__(256) gather_kernel(const uint4* __restrict__ pool, const int32_t* __restrict__ page_table,
                                                     int32_t n_tokens, uint4* __restrict__ out) {
    const int64_t total = int64_t(n_tokens) * kVecPerToken;
    for (int64_t i = blockIdx.x * int64_t(blockDim.x) + threadIdx.x; i < total; i += int64_t(gridDim.x) * blockDim.x) {
        const int32_t t = int32_t(i / kVecPerToken);
        const int32_t v = int32_t(i % kVecPerToken);
        const int64_t slot = int64_t(__ldg(page_table + t / kPage)) * kPage + t % kPage;
        out[i] = pool[slot * kVecPerToken + v];
    }
}

inline int grid_for(int64_t vecs, int sm_count) {
    int64_t blocks = (vecs + 255) / 256;
    int64_t cap = int64_t(sm_count) * 8;
    return int(blocks < 1 ? 1 : (blocks > cap ? cap : blocks));
}

}  // namespace

int launch_append(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens, const int32_t* page_table,
                  int32_t start_pos, cudaStream_t stream) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(unsigned(grid_for(int64_t(n_tokens) * kVecPerToken, ctx->sm_count)), 1, 1);
    cfg.blockDim = dim3(256, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    KAIROS_CUDA_TRY(cudaLaunchKernelEx(&cfg, append_kernel, reinterpret_cast<uint4*>(ctx->cfg.pool), reinterpret_cast<const uint4*>(latent),
                                       reinterpret_cast<const uint4*>(k_rope), page_table, n_tokens, start_pos));
    KAIROS_CUDA_TRY(cudaGetLastError());
    return KAIROS_OK;
}

int launch_append_decode(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n, const int32_t* page_tables,
                         int32_t table_stride, const int32_t* positions, cudaStream_t stream) {
    append_decode_kernel<<<grid_for(int64_t(n) * kVecPerToken, ctx->sm_count), 256, 0, stream>>>(
        reinterpret_cast<uint4*>(ctx->cfg.pool), reinterpret_cast<const uint4*>(latent),
        reinterpret_cast<const uint4*>(k_rope), page_tables, table_stride, positions, n);
    KAIROS_CUDA_TRY(cudaGetLastError());
    return KAIROS_OK;
}

int launch_gather(kairos_ctx* ctx, const int32_t* page_table, int32_t n_tokens, void* out, cudaStream_t stream) {
    gather_kernel<<<grid_for(int64_t(n_tokens) * kVecPerToken, ctx->sm_count), 256, 0, stream>>>(
        reinterpret_cast<const uint4*>(ctx->cfg.pool), page_table, n_tokens, reinterpret_cast<uint4*>(out));
    KAIROS_CUDA_TRY(cudaGetLastError());
    return KAIROS_OK;
}

}  // namespace kairos
