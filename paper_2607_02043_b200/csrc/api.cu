// C-ABI entry points of libkairos.so (include/kairos.h): argument validation, host planner, staging, launches.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include "kairos_internal.h"

namespace kairos {

static thread_local std::string g_last_error;

void set_error(const std::string& msg) { g_last_error = msg; }
int fail(int code, const std::string& msg) {
    g_last_error = msg;
    return code;
}

constexpr int kMaxCtas = 192;  // bound used by kairos_workspace_bytes (B200 has 148 SMs, one CTA each)
constexpr size_t kCounterBytes = 256;

static size_t max_partial_slots(int32_t max_decodes) { return size_t(std::max(0, max_decodes)) + 12 * size_t(kMaxCtas); }

int staging_acquire(kairos_ctx* ctx, size_t bytes, StagingSlot** out) {
    StagingSlot& s = ctx->staging[ctx->staging_next];
    ctx->staging_next = (ctx->staging_next + 1) % kairos_ctx::kStagingSlots;
    if (s.used) KAIROS_CUDA_TRY(cudaEventSynchronize(s.done));  // its last H2D copy has left the pinned buffer
    if (s.bytes < bytes) {
        if (s.host) cudaFreeHost(s.host);
        if (s.dev) cudaFree(s.dev);
        s.host = s.dev = nullptr;
        s.bytes = 0;
        size_t cap = std::max<size_t>(bytes * 2, 64 * 1024);
        KAIROS_CUDA_TRY(cudaMallocHost(&s.host, cap));
        KAIROS_CUDA_TRY(cudaMalloc(&s.dev, cap));
        s.bytes = cap;
    }
    if (!s.done) KAIROS_CUDA_TRY(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
    s.used = true;
    *out = &s;
    return KAIROS_OK;
}

static int check_ctx(const kairos_ctx* ctx) {
    if (!ctx) return fail(KAIROS_ERR_INVALID_ARG, "ctx is NULL");
    return KAIROS_OK;
}

// Shared by kairos_mixed_step and the latency table: validate, plan, stage, launch.
static int mixed_step_impl(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                           int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len,
                           const void* q_chunk, const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec,
                           void* out_chunk, float* lse_dec, float* lse_chunk, cudaStream_t stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n_dec < 0 || chunk_len < 0 || prefix_len < 0) return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    if (n_dec > 0) {
        if (!q_dec || !dec_page_tables || !dec_ctx_lens || !out_dec) return fail(KAIROS_ERR_INVALID_ARG, "NULL decode argument");
        if (dec_table_stride < 1) return fail(KAIROS_ERR_INVALID_ARG, "dec_table_stride < 1");
        for (int32_t i = 0; i < n_dec; ++i) {
            if (dec_ctx_lens[i] < 1) return fail(KAIROS_ERR_INVALID_ARG, "dec_ctx_lens[" + std::to_string(i) + "] < 1");
            if (int64_t(dec_ctx_lens[i]) > int64_t(dec_table_stride) * kPage)
                return fail(KAIROS_ERR_INVALID_ARG, "dec_ctx_lens[" + std::to_string(i) + "] beyond its page table");
        }
    }
    if (chunk_len > 0) {
        if (!q_chunk || !chunk_page_table || !out_chunk) return fail(KAIROS_ERR_INVALID_ARG, "NULL chunk argument");
        if (int64_t(prefix_len) + chunk_len > int64_t(chunk_table_len) * kPage)
            return fail(KAIROS_ERR_INVALID_ARG, "chunk page table shorter than prefix_len + chunk_len");
    }
    std::memset(ctx->last_info, 0, sizeof(ctx->last_info));
    if (n_dec == 0 && chunk_len == 0) return KAIROS_OK;

    StepArgs a{n_dec, q_dec, dec_page_tables, dec_table_stride, chunk_len, prefix_len,
               q_chunk, chunk_page_table, out_dec, out_chunk, lse_dec, lse_chunk};

    if (ctx->impl == 0) {
        StagingSlot* st = nullptr;
        if (int rc = staging_acquire(ctx, sizeof(int32_t) * size_t(std::max(n_dec, 1)), &st)) return rc;
        if (n_dec > 0) {
            std::memcpy(st->host, dec_ctx_lens, sizeof(int32_t) * size_t(n_dec));
            KAIROS_CUDA_TRY(cudaMemcpyAsync(st->dev, st->host, sizeof(int32_t) * size_t(n_dec), cudaMemcpyHostToDevice, stream));
        }
        KAIROS_CUDA_TRY(cudaEventRecord(st->done, stream));
        if (int rc = launch_attn_simple(ctx, a, reinterpret_cast<const int32_t*>(st->dev), stream)) return rc;
        ctx->last_info[0] = n_dec + chunk_len;
        ctx->last_info[3] = n_dec + chunk_len;
        ctx->last_info[4] = 1;
        return KAIROS_OK;
    }

    // ---- impl 1: plan -> staging -> persistent kernel (+ combine)
    static const bool dbg = std::getenv("KAIROS_DEBUG_TIMING") != nullptr;
    static double t_plan = 0, t_stage = 0, t_copy = 0, t_launch = 0; static long n_calls = 0;
    auto now = [] { return std::chrono::steady_clock::now(); };
    auto us = [](auto a, auto b) { return std::chrono::duration<double, std::micro>(b - a).count(); };
    auto T0 = now();
    Plan& plan = ctx->plan;
    build_plan(dec_ctx_lens, n_dec, chunk_len, prefix_len, umma_resident_ctas(ctx), umma_chunk_tile_tokens(), &plan,
               ctx->force_pairs, pair_tile_tokens());
    const size_t ws_needed = kCounterBytes + size_t(plan.n_partial_slots) * kPartialSlotBytes;
    if (ws_needed > ctx->cfg.workspace_bytes)
        return fail(KAIROS_ERR_WORKSPACE, "workspace too small: need " + std::to_string(ws_needed) + " bytes");
    const size_t items_bytes = plan.items.size() * sizeof(WorkItem);
    const size_t comb_bytes = plan.combines.size() * sizeof(CombineItem);
    const size_t comb_off = (items_bytes + 255) / 256 * 256;
    const size_t pair_bytes = plan.pair_items.size() * sizeof(WorkItem);
    const size_t pair_off = (comb_off + comb_bytes + 255) / 256 * 256;
    StagingSlot* st = nullptr;
    auto T1 = now();
    if (int rc = staging_acquire(ctx, pair_off + pair_bytes + 256, &st)) return rc;
    auto T2 = now();
    std::memcpy(st->host, plan.items.data(), items_bytes);
    if (comb_bytes) std::memcpy(static_cast<uint8_t*>(st->host) + comb_off, plan.combines.data(), comb_bytes);
    if (pair_bytes) std::memcpy(static_cast<uint8_t*>(st->host) + pair_off, plan.pair_items.data(), pair_bytes);
    // The work list goes to the device on the library's copy stream, so that it overlaps whatever the caller's stream is
    // still running (the append of this step, the previous step's tail); the caller's stream then waits for it.  The
    // slot's device buffer is not overwritten before the kernels of its previous use have read it (`consumed`).
    if (ctx->copy_stream) {
        if (st->consumed) KAIROS_CUDA_TRY(cudaStreamWaitEvent(ctx->copy_stream, st->consumed, 0));
        KAIROS_CUDA_TRY(cudaMemcpyAsync(st->dev, st->host, pair_off + pair_bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
        KAIROS_CUDA_TRY(cudaEventRecord(st->done, ctx->copy_stream));
        KAIROS_CUDA_TRY(cudaStreamWaitEvent(stream, st->done, 0));
    } else {
        KAIROS_CUDA_TRY(cudaMemcpyAsync(st->dev, st->host, pair_off + pair_bytes, cudaMemcpyHostToDevice, stream));
        KAIROS_CUDA_TRY(cudaEventRecord(st->done, stream));
    }
    auto T3 = now();
    int kernels = 0;
    // Roofline leg of bench.py: one pair of events around the attention kernels of the step (the decode grid and, when
    // the planner uses it, the concurrent pair grid; fork and join are inside the bracket).
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->profile) {
        if (ctx->prof_used + 2 > ctx->prof_events.size()) {
            for (int i = 0; i < 2; ++i) {
                cudaEvent_t e;
                KAIROS_CUDA_TRY(cudaEventCreate(&e));
                ctx->prof_events.push_back(e);
            }
        }
        e0 = ctx->prof_events[ctx->prof_used];
        e1 = ctx->prof_events[ctx->prof_used + 1];
        ctx->prof_used += 2;
        KAIROS_CUDA_TRY(cudaEventRecord(e0, stream));
    }
    const WorkItem* dev_pair = reinterpret_cast<const WorkItem*>(static_cast<uint8_t*>(st->dev) + pair_off);
    const int n_pairs = plan.n_pairs;
    const bool have_queue = !plan.items.empty();
    const WorkItem* dev_items = reinterpret_cast<const WorkItem*>(st->dev);
    const CombineItem* dev_comb = reinterpret_cast<const CombineItem*>(static_cast<uint8_t*>(st->dev) + comb_off);
    if (n_pairs > 0 && have_queue) {
        // The two grids share the SMs in time (plan.cpp::choose_pairs).  dec_ctas > 0: the decode grid goes first, as 2-CTA
        // clusters on dec_ctas SMs (whole TPCs), then one chunk cluster per SM pair -- those that do not fit yet start when
        // the decode CTAs exit.  dec_ctas == 0: the clusters take every SM pair and the decode CTAs follow as SMs free up.
        // Both kernels go to the caller's stream; the second one is launched with programmatic stream serialisation and
        // starts once every CTA of the first is resident (both trigger launch_dependents on entry), so the order in
        // which the grids take SMs is the launch order.
        if (plan.dec_ctas > 0) {
            if (int rc = launch_attn_umma(ctx, a, dev_items, int32_t(plan.items.size()), dev_comb, int32_t(plan.combines.size()), stream,
                                          &kernels, plan.dec_ctas, /*as_clusters=*/true, /*pdl=*/false))
                return rc;
            if (int rc = launch_attn_pair(ctx, a, dev_pair, int32_t(plan.pair_items.size()), n_pairs, stream, /*pdl=*/true)) return rc;
        } else {
            if (int rc = launch_attn_pair(ctx, a, dev_pair, int32_t(plan.pair_items.size()), n_pairs, stream, /*pdl=*/false)) return rc;
            if (int rc = launch_attn_umma(ctx, a, dev_items, int32_t(plan.items.size()), dev_comb, int32_t(plan.combines.size()), stream,
                                          &kernels, umma_resident_ctas(ctx), /*as_clusters=*/false, /*pdl=*/true))
                return rc;
        }
    } else if (n_pairs > 0) {
        if (int rc = launch_attn_pair(ctx, a, dev_pair, int32_t(plan.pair_items.size()), n_pairs, stream, /*pdl=*/false)) return rc;
    } else if (have_queue) {
        if (int rc = launch_attn_umma(ctx, a, dev_items, int32_t(plan.items.size()), dev_comb, int32_t(plan.combines.size()), stream,
                                      &kernels, umma_resident_ctas(ctx), /*as_clusters=*/false, /*pdl=*/false))
            return rc;
    }
    if (n_pairs > 0) ++kernels;
    if (e1) KAIROS_CUDA_TRY(cudaEventRecord(e1, stream));
    if (!plan.combines.empty()) {
        if (int rc = launch_combine(ctx, a, reinterpret_cast<const CombineItem*>(static_cast<uint8_t*>(st->dev) + comb_off),
                                    int32_t(plan.combines.size()), stream))
            return rc;
        ++kernels;
    }
    if (ctx->copy_stream) {
        if (!st->consumed) KAIROS_CUDA_TRY(cudaEventCreateWithFlags(&st->consumed, cudaEventDisableTiming));
        KAIROS_CUDA_TRY(cudaEventRecord(st->consumed, stream));
    }
    if (dbg) {
        auto T4 = now();
        t_plan += us(T0, T1); t_stage += us(T1, T2); t_copy += us(T2, T3); t_launch += us(T3, T4);
        if (++n_calls % 500 == 0)
            std::fprintf(stderr, "[kairos host us/call] plan %.1f staging_wait %.1f copy+record %.1f encode+launch %.1f\n",
                         t_plan / n_calls, t_stage / n_calls, t_copy / n_calls, t_launch / n_calls);
    }
    ctx->last_info[0] = int64_t(plan.items.size());
    ctx->last_info[1] = plan.n_decode_items;
    ctx->last_info[2] = plan.n_chunk_items + int64_t(plan.pair_items.size());
    ctx->last_info[3] = std::min<int64_t>(plan.n_pairs > 0 && plan.dec_ctas > 0 ? plan.dec_ctas : umma_resident_ctas(ctx), int64_t(plan.items.size()));
    ctx->last_info[4] = kernels;
    ctx->last_info[5] = int64_t(ws_needed);
    ctx->last_info[6] = plan.n_pairs;
    return KAIROS_OK;
}

}  // namespace kairos

using namespace kairos;

extern "C" {

size_t kairos_workspace_bytes(int32_t max_decodes, int32_t max_chunk) {
    (void)max_chunk;  // chunk tiles are KV-split only while they are fewer than the CTAs: bounded by kMaxCtas
    return kCounterBytes + max_partial_slots(max_decodes) * kPartialSlotBytes;
}

int kairos_create(const kairos_config* cfg, kairos_ctx** out) {
    if (!cfg || !out) return fail(KAIROS_ERR_INVALID_ARG, "cfg or out is NULL");
    if (cfg->num_heads != kHeads || cfg->latent_dim != kLatent || cfg->rope_dim != kRope || cfg->page_size != kPage)
        return fail(KAIROS_ERR_UNSUPPORTED, "only num_heads=16, latent_dim=512, rope_dim=64, page_size=64 are built");
    if (!(cfg->softmax_scale > 0.f) || !std::isfinite(cfg->softmax_scale))
        return fail(KAIROS_ERR_INVALID_ARG, "softmax_scale must be finite and > 0");
    if (!cfg->pool || cfg->num_pages < 1) return fail(KAIROS_ERR_INVALID_ARG, "pool is NULL or num_pages < 1");
    if (reinterpret_cast<uintptr_t>(cfg->pool) % 128) return fail(KAIROS_ERR_INVALID_ARG, "pool must be 128-byte aligned");
    if (cfg->workspace_bytes > 0 && (!cfg->workspace || reinterpret_cast<uintptr_t>(cfg->workspace) % 256))
        return fail(KAIROS_ERR_INVALID_ARG, "workspace must be non-NULL and 256-byte aligned");
    int n_dev = 0;
    KAIROS_CUDA_TRY(cudaGetDeviceCount(&n_dev));
    if (cfg->device < 0 || cfg->device >= n_dev) return fail(KAIROS_ERR_INVALID_ARG, "no such CUDA device");
    KAIROS_CUDA_TRY(cudaSetDevice(cfg->device));
    cudaDeviceProp prop;
    KAIROS_CUDA_TRY(cudaGetDeviceProperties(&prop, cfg->device));
    if (prop.major != 10) return fail(KAIROS_ERR_UNSUPPORTED, "libkairos is built for sm_100a (B200) only");
    kairos_ctx* ctx = new (std::nothrow) kairos_ctx();
    if (!ctx) return fail(KAIROS_ERR_INVALID_ARG, "out of host memory");
    ctx->cfg = *cfg;
    ctx->sm_count = prop.multiProcessorCount;
    const char* impl = std::getenv("KAIROS_IMPL");
    ctx->impl = (impl && std::string(impl) == "simple") ? 0 : 1;
    if (ctx->impl == 1) {
        if (cfg->workspace_bytes < kCounterBytes) {
            delete ctx;
            return fail(KAIROS_ERR_WORKSPACE, "workspace must hold at least 256 bytes (work-queue counters)");
        }
        if (int rc = umma_init(ctx)) {
            delete ctx;
            return rc;
        }
        if (int rc = pair_init(ctx)) {
            delete ctx;
            return rc;
        }
        if (!std::getenv("KAIROS_NO_COPY_STREAM")) KAIROS_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        if (const char* fp = std::getenv("KAIROS_PAIRS")) ctx->force_pairs = std::atoi(fp);  // debug / sweeps: 0 = gen-1 chunk tiles only
        if (const char* fd = std::getenv("KAIROS_DEC_ONLY")) ctx->force_dec_only = std::atoi(fd);
    }
    *out = ctx;
    return KAIROS_OK;
}

int kairos_destroy(kairos_ctx* ctx) {
    if (!ctx) return KAIROS_OK;
    cudaSetDevice(ctx->cfg.device);
    for (auto& s : ctx->staging) {
        if (s.used && s.done) cudaEventSynchronize(s.done);
        if (s.host) cudaFreeHost(s.host);
        if (s.dev) cudaFree(s.dev);
        if (s.done) cudaEventDestroy(s.done);
        if (s.consumed) cudaEventDestroy(s.consumed);
    }
    if (ctx->host_stage.dev) cudaFree(ctx->host_stage.dev);
    for (auto e : ctx->prof_events) cudaEventDestroy(e);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
    return KAIROS_OK;
}

int kairos_append_latent(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens,
                         const int32_t* page_table, int32_t table_len, int32_t start_pos, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n_tokens < 0 || start_pos < 0 || table_len < 0) return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    if (n_tokens == 0) return KAIROS_OK;
    if (!latent || !k_rope || !page_table) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    if (int64_t(start_pos) + n_tokens > int64_t(table_len) * kPage)
        return fail(KAIROS_ERR_INVALID_ARG, "start_pos + n_tokens beyond table_len*64");
    if (reinterpret_cast<uintptr_t>(latent) % 16 || reinterpret_cast<uintptr_t>(k_rope) % 16)
        return fail(KAIROS_ERR_INVALID_ARG, "latent / k_rope must be 16-byte aligned");
    return launch_append(ctx, latent, k_rope, n_tokens, page_table, start_pos, static_cast<cudaStream_t>(cuda_stream));
}

int kairos_append_decode_tokens(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n,
                                const int32_t* page_tables, int32_t table_stride, const int32_t* positions,
                                void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n < 0 || table_stride < 1) return fail(KAIROS_ERR_INVALID_ARG, "n < 0 or table_stride < 1");
    if (n == 0) return KAIROS_OK;
    if (!latent || !k_rope || !page_tables || !positions) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    if (reinterpret_cast<uintptr_t>(latent) % 16 || reinterpret_cast<uintptr_t>(k_rope) % 16)
        return fail(KAIROS_ERR_INVALID_ARG, "latent / k_rope must be 16-byte aligned");
    return launch_append_decode(ctx, latent, k_rope, n, page_tables, table_stride, positions,
                                static_cast<cudaStream_t>(cuda_stream));
}

int kairos_gather_latent(kairos_ctx* ctx, const int32_t* page_table, int32_t table_len, int32_t n_tokens, void* out,
                         void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n_tokens < 0 || table_len < 0) return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    if (n_tokens == 0) return KAIROS_OK;
    if (!page_table || !out) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    if (int64_t(n_tokens) > int64_t(table_len) * kPage) return fail(KAIROS_ERR_INVALID_ARG, "n_tokens beyond table_len*64");
    if (reinterpret_cast<uintptr_t>(out) % 16) return fail(KAIROS_ERR_INVALID_ARG, "out must be 16-byte aligned");
    return launch_gather(ctx, page_table, n_tokens, out, static_cast<cudaStream_t>(cuda_stream));
}

int kairos_mixed_step(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                      int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len,
                      const void* q_chunk, const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec,
                      void* out_chunk, float* lse_dec, float* lse_chunk, void* cuda_stream) {
    return mixed_step_impl(ctx, n_dec, q_dec, dec_page_tables, dec_table_stride, dec_ctx_lens, chunk_len, prefix_len,
                           q_chunk, chunk_page_table, chunk_table_len, out_dec, out_chunk, lse_dec, lse_chunk,
                           static_cast<cudaStream_t>(cuda_stream));
}

int kairos_mixed_step_host(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                           int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len,
                           int32_t prefix_len, const void* q_chunk, const void* chunk_latent, const void* chunk_k_rope,
                           const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec, void* out_chunk,
                           float* lse_dec, float* lse_chunk, uint64_t* h2d_bytes, uint64_t* d2h_bytes,
                           void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n_dec < 0 || chunk_len < 0 || prefix_len < 0 || dec_table_stride < 0 || chunk_table_len < 0)
        return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    if (n_dec > 0 && (!q_dec || !dec_page_tables || !dec_ctx_lens || !out_dec))
        return fail(KAIROS_ERR_INVALID_ARG, "NULL decode argument");
    if (chunk_len > 0 && (!q_chunk || !chunk_latent || !chunk_k_rope || !chunk_page_table || !out_chunk))
        return fail(KAIROS_ERR_INVALID_ARG, "NULL chunk argument");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    const size_t b_qd = al(size_t(n_dec) * kHeads * kDim * 2), b_qc = al(size_t(chunk_len) * kHeads * kDim * 2);
    const size_t b_dpt = al(size_t(n_dec) * dec_table_stride * 4), b_cpt = al(size_t(chunk_table_len) * 4);
    const size_t b_lat = al(size_t(chunk_len) * kLatent * 2), b_rope = al(size_t(chunk_len) * kRope * 2);
    const size_t b_od = al(size_t(n_dec) * kHeads * kLatent * 2), b_oc = al(size_t(chunk_len) * kHeads * kLatent * 2);
    const size_t b_ld = al(size_t(n_dec) * kHeads * 4), b_lc = al(size_t(chunk_len) * kHeads * 4);
    const size_t total = b_qd + b_qc + b_dpt + b_cpt + b_lat + b_rope + b_od + b_oc + b_ld + b_lc;
    if (ctx->host_stage.bytes < total) {
        KAIROS_CUDA_TRY(cudaStreamSynchronize(stream));
        if (ctx->host_stage.dev) cudaFree(ctx->host_stage.dev);
        ctx->host_stage.dev = nullptr;
        ctx->host_stage.bytes = 0;
        KAIROS_CUDA_TRY(cudaMalloc(&ctx->host_stage.dev, total));
        ctx->host_stage.bytes = total;
    }
    uint8_t* p = static_cast<uint8_t*>(ctx->host_stage.dev);
    uint8_t* d_qd = p;  p += b_qd;
    uint8_t* d_qc = p;  p += b_qc;
    uint8_t* d_dpt = p; p += b_dpt;
    uint8_t* d_cpt = p; p += b_cpt;
    uint8_t* d_lat = p; p += b_lat;
    uint8_t* d_rope = p; p += b_rope;
    uint8_t* d_od = p;  p += b_od;
    uint8_t* d_oc = p;  p += b_oc;
    uint8_t* d_ld = p;  p += b_ld;
    uint8_t* d_lc = p;
    uint64_t h2d = 0, d2h = 0;
    auto up = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!bytes) return cudaSuccess;
        h2d += bytes;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);
    };
    auto down = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!bytes || !dst) return cudaSuccess;
        d2h += bytes;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, stream);
    };
    KAIROS_CUDA_TRY(up(d_qd, q_dec, size_t(n_dec) * kHeads * kDim * 2));
    KAIROS_CUDA_TRY(up(d_dpt, dec_page_tables, size_t(n_dec) * dec_table_stride * 4));
    KAIROS_CUDA_TRY(up(d_qc, q_chunk, size_t(chunk_len) * kHeads * kDim * 2));
    KAIROS_CUDA_TRY(up(d_cpt, chunk_page_table, size_t(chunk_len > 0 ? chunk_table_len : 0) * 4));
    KAIROS_CUDA_TRY(up(d_lat, chunk_latent, size_t(chunk_len) * kLatent * 2));
    KAIROS_CUDA_TRY(up(d_rope, chunk_k_rope, size_t(chunk_len) * kRope * 2));
    if (chunk_len > 0) {
        if (int rc = kairos_append_latent(ctx, d_lat, d_rope, chunk_len, reinterpret_cast<const int32_t*>(d_cpt),
                                          chunk_table_len, prefix_len, cuda_stream))
            return rc;
    }
    if (int rc = mixed_step_impl(ctx, n_dec, d_qd, reinterpret_cast<const int32_t*>(d_dpt), dec_table_stride,
                                 dec_ctx_lens, chunk_len, prefix_len, d_qc, reinterpret_cast<const int32_t*>(d_cpt),
                                 chunk_table_len, d_od, d_oc, lse_dec ? reinterpret_cast<float*>(d_ld) : nullptr,
                                 lse_chunk ? reinterpret_cast<float*>(d_lc) : nullptr, stream))
        return rc;
    KAIROS_CUDA_TRY(down(out_dec, d_od, size_t(n_dec) * kHeads * kLatent * 2));
    KAIROS_CUDA_TRY(down(out_chunk, d_oc, size_t(chunk_len) * kHeads * kLatent * 2));
    KAIROS_CUDA_TRY(down(lse_dec, d_ld, size_t(n_dec) * kHeads * 4));
    KAIROS_CUDA_TRY(down(lse_chunk, d_lc, size_t(chunk_len) * kHeads * 4));
    KAIROS_CUDA_TRY(cudaStreamSynchronize(stream));
    if (h2d_bytes) *h2d_bytes = h2d;
    if (d2h_bytes) *d2h_bytes = d2h;
    return KAIROS_OK;
}

int kairos_plan_dump(const int32_t* dec_ctx_lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len, int32_t n_ctas,
                     int32_t pair_mode, int32_t* items_out, int32_t max_items, int32_t* n_items_out,
                     int32_t* n_partial_slots_out, int32_t* n_pairs_out) {
    if (n_dec < 0 || chunk_len < 0 || prefix_len < 0 || n_ctas < 1 || max_items < 0 || !n_items_out)
        return fail(KAIROS_ERR_INVALID_ARG, "bad size or NULL n_items_out");
    if (n_dec > 0 && !dec_ctx_lens) return fail(KAIROS_ERR_INVALID_ARG, "dec_ctx_lens is NULL");
    for (int32_t i = 0; i < n_dec; ++i)
        if (dec_ctx_lens[i] < 1) return fail(KAIROS_ERR_INVALID_ARG, "dec_ctx_lens[" + std::to_string(i) + "] < 1");
    Plan plan;
    build_plan(dec_ctx_lens, n_dec, chunk_len, prefix_len, n_ctas, umma_chunk_tile_tokens(), &plan, pair_mode, pair_tile_tokens());
    for (WorkItem w : plan.pair_items) {  // appended after the queue, marked kind 2
        w.kind = 2;
        plan.items.push_back(w);
    }
    if (n_pairs_out) *n_pairs_out = plan.n_pairs;
    *n_items_out = int32_t(plan.items.size());
    if (n_partial_slots_out) *n_partial_slots_out = plan.n_partial_slots;
    if (items_out)
        std::memcpy(items_out, plan.items.data(), sizeof(WorkItem) * size_t(std::min<int64_t>(max_items, int64_t(plan.items.size()))));
    return KAIROS_OK;
}

int kairos_last_plan_info(const kairos_ctx* ctx, int64_t* info, int32_t n) {
    if (!ctx || !info || n < 0) return fail(KAIROS_ERR_INVALID_ARG, "NULL argument");
    for (int32_t i = 0; i < n && i < 7; ++i) info[i] = ctx->last_info[i];
    return KAIROS_OK;
}

int kairos_profile_enable(kairos_ctx* ctx, int32_t on) {
    if (int rc = check_ctx(ctx)) return rc;
    ctx->profile = on != 0;
    return KAIROS_OK;
}

int kairos_profile_read(kairos_ctx* ctx, double* main_kernel_us_total, int64_t* launches) {
    if (int rc = check_ctx(ctx)) return rc;
    double total = 0.0;
    for (size_t i = 0; i + 1 < ctx->prof_used; i += 2) {
        KAIROS_CUDA_TRY(cudaEventSynchronize(ctx->prof_events[i + 1]));
        float ms = 0.f;
        KAIROS_CUDA_TRY(cudaEventElapsedTime(&ms, ctx->prof_events[i], ctx->prof_events[i + 1]));
        total += double(ms) * 1e3;
    }
    if (main_kernel_us_total) *main_kernel_us_total = total;
    if (launches) *launches = int64_t(ctx->prof_used / 2);
    ctx->prof_used = 0;
    return KAIROS_OK;
}

const char* kairos_last_error(void) { return g_last_error.c_str(); }

const char* kairos_version(void) { return "kairos-b200 sm_100a gen1 (tcgen05 swapped-operand split-KV + persistent work queue)"; }

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// a11: latency table
// ---------------------------------------------------------------------------------------------------------------
namespace kairos {
namespace {

__global__ void fill_q_kernel(uint16_t* q, size_t n, uint32_t seed) {
    // cheap counter hash -> bf16 values roughly uniform in [-0.17, 0.17] (std ~0.1 like the generators' q)
    for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < n; i += size_t(gridDim.x) * blockDim.x) {
        uint32_t x = uint32_t(i) * 2654435761u + seed;
        x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
        float f = (float(x >> 8) * (1.0f / 16777216.0f) - 0.5f) * 0.34f;
        q[i] = uint16_t(__float_as_uint(f) >> 16);
    }
}

__global__ void flush_kernel(uint4* buf, size_t n, uint32_t v) {
    for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < n; i += size_t(gridDim.x) * blockDim.x)
        buf[i] = make_uint4(v, v, v, v);
}

struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
};

}  // namespace
}  // namespace kairos

extern "C" int kairos_step_latency_table(kairos_ctx* ctx, const int32_t* Bs, int32_t nB, const int32_t* Ks, int32_t nK,
                                         const int32_t* Cs, int32_t nC, int32_t prefix_len, int32_t warmup, int32_t reps,
                                         int32_t flush_l2, double* out_median_us, double* out_min_us, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!Bs || !Ks || !Cs || !out_median_us || nB < 1 || nK < 1 || nC < 1 || prefix_len < 0 || warmup < 0 || reps < 1)
        return fail(KAIROS_ERR_INVALID_ARG, "bad latency-table argument");
    int32_t maxB = 0, maxK = 0, maxC = 0;
    for (int i = 0; i < nB; ++i) { if (Bs[i] < 0) return fail(KAIROS_ERR_INVALID_ARG, "B < 0"); maxB = std::max(maxB, Bs[i]); }
    for (int i = 0; i < nK; ++i) { if (Ks[i] < 1) return fail(KAIROS_ERR_INVALID_ARG, "K < 1"); maxK = std::max(maxK, Ks[i]); }
    for (int i = 0; i < nC; ++i) { if (Cs[i] < 0) return fail(KAIROS_ERR_INVALID_ARG, "C < 0"); maxC = std::max(maxC, Cs[i]); }
    const int64_t max_dec_pages = int64_t(maxB) * ((maxK + kPage - 1) / kPage);
    const int64_t max_chunk_pages = (int64_t(prefix_len) + maxC + kPage - 1) / kPage;
    if (max_dec_pages + max_chunk_pages > ctx->cfg.num_pages)
        return fail(KAIROS_ERR_WORKSPACE, "pool has too few pages for the largest grid point: need " +
                                              std::to_string(max_dec_pages + max_chunk_pages));
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    KAIROS_CUDA_TRY(cudaSetDevice(ctx->cfg.device));
    const int32_t stride = std::max(1, (maxK + kPage - 1) / kPage);
    DevBuf q_dec, q_chunk, o_dec, o_chunk, dpt, cpt, flush;
    const size_t nqd = size_t(std::max(maxB, 1)) * kHeads * kDim, nqc = size_t(std::max(maxC, 1)) * kHeads * kDim;
    KAIROS_CUDA_TRY(cudaMalloc(&q_dec.p, nqd * 2));
    KAIROS_CUDA_TRY(cudaMalloc(&q_chunk.p, nqc * 2));
    KAIROS_CUDA_TRY(cudaMalloc(&o_dec.p, size_t(std::max(maxB, 1)) * kHeads * kLatent * 2));
    KAIROS_CUDA_TRY(cudaMalloc(&o_chunk.p, size_t(std::max(maxC, 1)) * kHeads * kLatent * 2));
    KAIROS_CUDA_TRY(cudaMalloc(&dpt.p, size_t(std::max(maxB, 1)) * stride * 4));
    KAIROS_CUDA_TRY(cudaMalloc(&cpt.p, size_t(std::max<int64_t>(max_chunk_pages, 1)) * 4));
    const size_t flush_bytes = size_t(256) << 20;  // > 126 MB L2
    if (flush_l2) KAIROS_CUDA_TRY(cudaMalloc(&flush.p, flush_bytes));
    fill_q_kernel<<<256, 256, 0, stream>>>(static_cast<uint16_t*>(q_dec.p), nqd, 0x1234u);
    fill_q_kernel<<<256, 256, 0, stream>>>(static_cast<uint16_t*>(q_chunk.p), nqc, 0x9876u);
    KAIROS_CUDA_TRY(cudaGetLastError());
    cudaEvent_t e0, e1;
    KAIROS_CUDA_TRY(cudaEventCreate(&e0));
    KAIROS_CUDA_TRY(cudaEventCreate(&e1));
    std::vector<int32_t> h_dpt, h_cpt, lens;
    std::vector<double> times;
    int rc = KAIROS_OK;
    for (int iB = 0; iB < nB && rc == KAIROS_OK; ++iB)
        for (int iK = 0; iK < nK && rc == KAIROS_OK; ++iK)
            for (int iC = 0; iC < nC && rc == KAIROS_OK; ++iC) {
                const int32_t B = Bs[iB], K = Ks[iK], C = Cs[iC];
                const size_t o = (size_t(iB) * nK + iK) * nC + iC;
                if (B == 0 && C == 0) { out_median_us[o] = 0.0; if (out_min_us) out_min_us[o] = 0.0; continue; }
                // distinct pages, strided through the pool (an odd multiplicative step visits each page once)
                const int64_t kp = (K + kPage - 1) / kPage, cp = C > 0 ? (int64_t(prefix_len) + C + kPage - 1) / kPage : 0;
                const int64_t need = int64_t(B) * kp + cp, np = ctx->cfg.num_pages;
                int64_t step = (np / 2) | 1;
                while (std::gcd(step, np) != 1) step += 2;
                auto page_of = [&](int64_t i) { return int32_t((i * step) % np); };
                (void)need;
                h_dpt.assign(size_t(std::max(B, 1)) * stride, 0);
                for (int64_t b = 0; b < B; ++b)
                    for (int64_t p = 0; p < kp; ++p) h_dpt[size_t(b) * stride + p] = page_of(b * kp + p);
                h_cpt.assign(size_t(std::max<int64_t>(cp, 1)), 0);
                for (int64_t p = 0; p < cp; ++p) h_cpt[size_t(p)] = page_of(int64_t(B) * kp + p);
                lens.assign(size_t(std::max(B, 1)), K);
                cudaMemcpyAsync(dpt.p, h_dpt.data(), h_dpt.size() * 4, cudaMemcpyHostToDevice, stream);
                cudaMemcpyAsync(cpt.p, h_cpt.data(), h_cpt.size() * 4, cudaMemcpyHostToDevice, stream);
                cudaStreamSynchronize(stream);
                times.clear();
                for (int it = 0; it < warmup + reps && rc == KAIROS_OK; ++it) {
                    if (flush_l2) flush_kernel<<<1184, 256, 0, stream>>>(static_cast<uint4*>(flush.p), flush_bytes / 16, uint32_t(it));
                    cudaEventRecord(e0, stream);
                    rc = mixed_step_impl(ctx, B, q_dec.p, static_cast<int32_t*>(dpt.p), stride, lens.data(), C, prefix_len,
                                         q_chunk.p, static_cast<int32_t*>(cpt.p), int32_t(std::max<int64_t>(cp, 1)), o_dec.p,
                                         o_chunk.p, nullptr, nullptr, stream);
                    cudaEventRecord(e1, stream);
                    if (cudaEventSynchronize(e1) != cudaSuccess) rc = fail(KAIROS_ERR_CUDA, "latency table: step failed on the device");
                    float ms = 0.f;
                    cudaEventElapsedTime(&ms, e0, e1);
                    if (it >= warmup) times.push_back(double(ms) * 1e3);
                }
                if (rc != KAIROS_OK) break;
                std::sort(times.begin(), times.end());
                const size_t n = times.size();
                out_median_us[o] = n % 2 ? times[n / 2] : 0.5 * (times[n / 2 - 1] + times[n / 2]);
                if (out_min_us) out_min_us[o] = times[0];
            }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc == KAIROS_OK) {
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(KAIROS_ERR_CUDA, std::string("latency table: ") + cudaGetErrorString(e));
    }
    return rc;
}
