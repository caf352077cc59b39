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

static int check_ctx(const kairos_ctx* ctx) {
    if (!ctx) return fail(KAIROS_ERR_INVALID_ARG, "ctx is NULL");
    return KAIROS_OK;
}

// Shape key of a step for the tuned launch orders: what the planner's decision depends on at page granularity.
static uint64_t shape_key(const int32_t* lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len) {
    uint64_t h = 1469598103934665603ull;
    auto mix = [&](uint64_t v) { h = (h ^ v) * 1099511628211ull; };
    mix(uint64_t(n_dec));
    for (int32_t i = 0; i < n_dec; ++i) mix(uint64_t((lens[i] + kPage - 1) / kPage));
    mix(uint64_t(chunk_len));
    mix(uint64_t((prefix_len + kPage - 1) / kPage));
    return h;
}

// The launch order the planner is asked for: the test knob if set, else what kairos_tune_step measured for this shape, else -1 (decide).
static int32_t pair_mode_for(const kairos_ctx* ctx, const int32_t* lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len) {
    if (ctx->force_pairs != -1 || ctx->tuned.empty() || chunk_len == 0) return ctx->force_pairs;
    const uint64_t k = shape_key(lens, n_dec, chunk_len, prefix_len);
    for (const TunedShape& t : ctx->tuned)
        if (t.key == k) return t.pair_mode;
    return -1;
}

static bool same_args(const StepArgs& a, const StepArgs& b) {
    return a.n_dec == b.n_dec && a.q_dec == b.q_dec && a.dec_page_tables == b.dec_page_tables &&
           a.dec_table_stride == b.dec_table_stride && a.chunk_len == b.chunk_len && a.prefix_len == b.prefix_len &&
           a.q_chunk == b.q_chunk && a.chunk_page_table == b.chunk_page_table && a.out_dec == b.out_dec &&
           a.out_chunk == b.out_chunk && a.lse_dec == b.lse_dec && a.lse_chunk == b.lse_chunk && a.fp8 == b.fp8;
}

static void drop_graph(PlanBuffer& b) {
    if (b.exec) cudaGraphExecDestroy(b.exec);
    b.exec = nullptr;
    b.same_args_uses = 0;
}

// Plan -> byte layout of its device copy: items | combines | pair items (256-byte aligned sections).
static void layout_entry(PlanEntry& e) {
    e.items_bytes = e.plan.items.size() * sizeof(WorkItem);
    e.comb_bytes = e.plan.combines.size() * sizeof(CombineItem);
    e.comb_off = (e.items_bytes + 255) / 256 * 256;
    e.pair_bytes = e.plan.pair_items.size() * sizeof(WorkItem);
    e.pair_off = (e.comb_off + e.comb_bytes + 255) / 256 * 256;
    e.total_bytes = e.pair_off + e.pair_bytes;
}

// Copies the entry's plan into buffer `bi` and sends it to the device.  The copy runs on the context's copy stream so that it
// overlaps whatever the caller's stream is still running (this step's append, the previous step's tail); the caller's stream
// waits for it.  The buffer's previous contents may still be read by kernels of an earlier step (`last_use`) and its pinned
// source by an earlier copy (`uploaded`): both are waited for, the first on the device, the second on the host (it completed
// long ago unless the host runs several steps ahead of the GPU).
static int upload_plan(kairos_ctx* ctx, PlanEntry& e, int bi, cudaStream_t stream) {
    PlanBuffer& b = e.buf[bi];
    const size_t need = e.total_bytes + 256;
    if (b.ever_used && b.uploaded) KAIROS_CUDA_TRY(cudaEventSynchronize(b.uploaded));
    if (b.cap < need) {
        if (b.ever_used && b.last_use) KAIROS_CUDA_TRY(cudaEventSynchronize(b.last_use));  // rare: the buffer grows
        drop_graph(b);  // it holds the old device pointer
        if (b.host) cudaFreeHost(b.host);
        if (b.dev) cudaFree(b.dev);
        b.host = b.dev = nullptr;
        b.cap = 0;
        const size_t cap = std::max<size_t>(need * 2, 64 * 1024);
        KAIROS_CUDA_TRY(cudaMallocHost(&b.host, cap));
        KAIROS_CUDA_TRY(cudaMalloc(&b.dev, cap));
        b.cap = cap;
    }
    if (!b.uploaded) KAIROS_CUDA_TRY(cudaEventCreateWithFlags(&b.uploaded, cudaEventDisableTiming));
    if (!b.last_use) KAIROS_CUDA_TRY(cudaEventCreateWithFlags(&b.last_use, cudaEventDisableTiming));
    uint8_t* h = static_cast<uint8_t*>(b.host);
    std::memcpy(h, e.plan.items.data(), e.items_bytes);
    if (e.comb_bytes) std::memcpy(h + e.comb_off, e.plan.combines.data(), e.comb_bytes);
    if (e.pair_bytes) std::memcpy(h + e.pair_off, e.plan.pair_items.data(), e.pair_bytes);
    cudaStream_t cs = (ctx->use_copy_stream && ctx->copy_stream) ? ctx->copy_stream : stream;
    if (b.ever_used && cs != stream) KAIROS_CUDA_TRY(cudaStreamWaitEvent(cs, b.last_use, 0));
    KAIROS_CUDA_TRY(cudaMemcpyAsync(b.dev, b.host, e.total_bytes, cudaMemcpyHostToDevice, cs));
    KAIROS_CUDA_TRY(cudaEventRecord(b.uploaded, cs));
    b.upload_pending = cs != stream;
    b.ever_used = true;
    return KAIROS_OK;
}

// The kernels of one step, in the order plan.cpp::choose_pairs decided, on `stream` (the caller's, or the capture stream).
static int launch_step_kernels(kairos_ctx* ctx, const PlanEntry& e, const PlanBuffer& b, const StepArgs& a, cudaStream_t stream,
                               cudaEvent_t e0, cudaEvent_t e1) {
    const Plan& plan = e.plan;
    const uint8_t* dev = static_cast<const uint8_t*>(b.dev);
    const WorkItem* dev_items = reinterpret_cast<const WorkItem*>(dev);
    const CombineItem* dev_comb = reinterpret_cast<const CombineItem*>(dev + e.comb_off);
    const WorkItem* dev_pair = reinterpret_cast<const WorkItem*>(dev + e.pair_off);
    const int n_items = int32_t(plan.items.size()), n_pair_items = int32_t(plan.pair_items.size());
    const int n_pairs = plan.n_pairs;
    const bool have_queue = n_items > 0;
    // Roofline leg of bench.py: one pair of events around the attention kernels of the step (the decode grid and, when the
    // planner uses it, the concurrent pair grid).
    if (e0) KAIROS_CUDA_TRY(cudaEventRecord(e0, stream));
    if (a.fp8) {
        if (int rc = launch_fp8_decode(ctx, a, dev_items, n_items, stream)) return rc;
    } else if (n_pairs > 0 && have_queue) {
        // The two grids share the SMs in time (plan.cpp::choose_pairs).  dec_ctas > 0: the decode grid goes first, as 2-CTA
        // clusters on dec_ctas SMs (whole TPCs), then one chunk cluster per SM pair -- those that do not fit yet start when
        // the decode CTAs exit.  dec_ctas == 0: the clusters go first and the decode CTAs follow as SMs free up.  The second
        // kernel is launched with programmatic stream serialisation and starts once every CTA of the first is resident (both
        // trigger launch_dependents on entry), so the order in which the grids take SMs is the launch order.
        if (plan.dec_ctas > 0) {
            if (int rc = launch_attn_umma(ctx, plan, a, dev_items, n_items, stream, plan.dec_ctas, /*as_clusters=*/true, /*pdl=*/false)) return rc;
            if (int rc = launch_attn_pair(ctx, a, dev_pair, n_pair_items, n_pairs, stream, /*pdl=*/true)) return rc;
        } else {
            if (int rc = launch_attn_pair(ctx, a, dev_pair, n_pair_items, n_pairs, stream, /*pdl=*/false)) return rc;
            if (int rc = launch_attn_umma(ctx, plan, a, dev_items, n_items, stream, umma_resident_ctas(ctx), /*as_clusters=*/false, /*pdl=*/true)) return rc;
        }
    } else if (n_pairs > 0) {
        if (int rc = launch_attn_pair(ctx, a, dev_pair, n_pair_items, n_pairs, stream, /*pdl=*/false)) return rc;
    } else if (have_queue) {
        if (int rc = launch_attn_umma(ctx, plan, a, dev_items, n_items, stream, umma_resident_ctas(ctx), /*as_clusters=*/false, /*pdl=*/false)) return rc;
    }
    if (e1) KAIROS_CUDA_TRY(cudaEventRecord(e1, stream));
    if (!plan.combines.empty())
        if (int rc = launch_combine(ctx, a, dev_comb, int32_t(plan.combines.size()), stream)) return rc;
    return KAIROS_OK;
}

// kairos_profile_enable: the next pair of events that brackets a step's attention kernels (NULL, NULL when profiling is off)
static int next_profile_events(kairos_ctx* ctx, cudaEvent_t* e0, cudaEvent_t* e1) {
    *e0 = *e1 = nullptr;
    if (!ctx->profile) return KAIROS_OK;
    if (ctx->prof_used + 2 > ctx->prof_events.size()) {
        for (int i = 0; i < 2; ++i) {
            cudaEvent_t ev;
            KAIROS_CUDA_TRY(cudaEventCreate(&ev));
            ctx->prof_events.push_back(ev);
        }
    }
    *e0 = ctx->prof_events[ctx->prof_used];
    *e1 = ctx->prof_events[ctx->prof_used + 1];
    ctx->prof_used += 2;
    return KAIROS_OK;
}

static int kernels_of(const Plan& plan) {
    return (plan.n_pairs > 0 ? 1 : 0) + (plan.items.empty() ? 0 : 1) + (plan.combines.empty() ? 0 : 1);
}

// Captures the step's launches (programmatic edges included) on the context's capture stream.  A failure is not an error of
// the step: graphs are switched off for this context and the caller launches directly.
static bool capture_graph(kairos_ctx* ctx, const PlanEntry& e, PlanBuffer& b, const StepArgs& a) {
    drop_graph(b);
    if (!ctx->capture_stream) return false;
    if (cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        ctx->use_graph = 0;
        return false;
    }
    const int rc = launch_step_kernels(ctx, e, b, a, ctx->capture_stream, nullptr, nullptr);
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(ctx->capture_stream, &graph);
    cudaGraphExec_t exec = nullptr;
    bool ok = rc == KAIROS_OK && ce == cudaSuccess && graph != nullptr;
    if (ok) ok = cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    if (!ok) {
        cudaGetLastError();
        if (exec) cudaGraphExecDestroy(exec);
        ctx->use_graph = 0;
        return false;
    }
    b.exec = exec;
    b.gargs = a;
    return true;
}

int mixed_step_impl(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                    int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len,
                    const void* q_chunk, const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec,
                    void* out_chunk, float* lse_dec, float* lse_chunk, cudaStream_t stream, int32_t fp8) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n_dec < 0 || chunk_len < 0 || prefix_len < 0) return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    auto misaligned = [](const void* p, uintptr_t a) { return reinterpret_cast<uintptr_t>(p) % a != 0; };
    if (n_dec > 0) {
        if (!q_dec || !dec_page_tables || !dec_ctx_lens || !out_dec) return fail(KAIROS_ERR_INVALID_ARG, "NULL decode argument");
        if (dec_table_stride < 1) return fail(KAIROS_ERR_INVALID_ARG, "dec_table_stride < 1");
        if (misaligned(q_dec, 16) || misaligned(out_dec, 16) || misaligned(lse_dec, 4) || misaligned(dec_page_tables, 4))
            return fail(KAIROS_ERR_INVALID_ARG, "q_dec / out_dec must be 16-byte aligned (lse_dec, page tables: 4)");
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
        if (misaligned(q_chunk, 16) || misaligned(out_chunk, 16) || misaligned(lse_chunk, 4) || misaligned(chunk_page_table, 4))
            return fail(KAIROS_ERR_INVALID_ARG, "q_chunk / out_chunk must be 16-byte aligned (lse_chunk, page table: 4)");
    }
    std::memset(ctx->last_info, 0, sizeof(ctx->last_info));
    if (n_dec == 0 && chunk_len == 0) return KAIROS_OK;

    const StepArgs a{n_dec, q_dec, dec_page_tables, dec_table_stride, chunk_len, prefix_len,
                     q_chunk, chunk_page_table, out_dec, out_chunk, lse_dec, lse_chunk, fp8};
    const int32_t target_ctas = umma_resident_ctas(ctx);
    const int32_t pair_mode = fp8 ? 0 : pair_mode_for(ctx, dec_ctx_lens, n_dec, chunk_len, prefix_len);

    // ---- a0: find the plan (exact hit: same lengths; structural hit: same page count per request), else build it
    PlanEntry* hit = nullptr;
    PlanEntry* structural = nullptr;
    PlanEntry* victim = &ctx->plans[ctx->plan_clock % kairos_ctx::kPlanEntries];  // cache off: rotate, so that a step's plan
                                                                                   // copy never waits for the previous step
    if (ctx->use_plan_cache) {
        victim = &ctx->plans[0];
        for (PlanEntry& e : ctx->plans) {
            if (!e.valid) { if (victim->valid) victim = &e; continue; }
            if (victim->valid && e.stamp < victim->stamp) victim = &e;
            if (e.n_dec != n_dec || e.chunk_len != chunk_len || e.prefix_len != prefix_len || e.target_ctas != target_ctas ||
                e.pair_mode != pair_mode || e.fp8 != fp8)
                continue;
            if (n_dec == 0 || std::memcmp(e.lens.data(), dec_ctx_lens, sizeof(int32_t) * size_t(n_dec)) == 0) { hit = &e; break; }
            if (!structural) {
                bool same = true;
                for (int32_t i = 0; i < n_dec && same; ++i) same = (e.lens[i] + kPage - 1) / kPage == (dec_ctx_lens[i] + kPage - 1) / kPage;
                if (same) structural = &e;
            }
        }
    }
    int cache_state = 0;  // 0 miss, 1 structural hit, 2 exact hit
    PlanEntry* e = hit;
    if (hit) {
        cache_state = 2;
    } else if (structural) {
        // only n_keys of the decode items moves with the lengths (plan.cpp never looks below page granularity)
        e = structural;
        cache_state = 1;
        e->lens.assign(dec_ctx_lens, dec_ctx_lens + n_dec);
        for (WorkItem& w : e->plan.items)
            if (w.kind == 0 && w.q_index < n_dec) w.n_keys = dec_ctx_lens[w.q_index];  // (fp8: q_index >= n_dec is a chunk token)
        e->cur ^= 1;
        if (int rc = upload_plan(ctx, *e, e->cur, stream)) return rc;
    } else {
        e = victim;
        for (PlanBuffer& b : e->buf) drop_graph(b);
        e->valid = false;
        if (fp8 && chunk_len > 0) {
            // the fp8 kernel has no chunk tiles: token j of the chunk runs as a one-token request over the chunk's own sequence
            // (n_keys = P + j + 1), planned with the decodes; its items and combine entries are mapped to the chunk's buffers
            std::vector<int32_t> all(dec_ctx_lens, dec_ctx_lens + n_dec);
            for (int32_t j = 0; j < chunk_len; ++j) all.push_back(prefix_len + j + 1);
            build_plan(all.data(), n_dec + chunk_len, 0, 0, target_ctas, umma_chunk_tile_tokens(), &e->plan, 0, pair_tile_tokens());
            for (CombineItem& c : e->plan.combines)
                if (c.q_index >= n_dec) {
                    c.q_index -= n_dec;
                    c.kind_stride |= 1;  // output rows of the chunk
                }
        } else {
            build_plan(dec_ctx_lens, n_dec, chunk_len, prefix_len, target_ctas, umma_chunk_tile_tokens(), &e->plan, pair_mode, pair_tile_tokens());
        }
        const size_t ws_needed = kCounterBytes + size_t(e->plan.n_partial_slots) * kPartialSlotBytes;
        if (ws_needed > ctx->cfg.workspace_bytes)
            return fail(KAIROS_ERR_WORKSPACE, "workspace too small: need " + std::to_string(ws_needed) + " bytes");
        e->n_dec = n_dec; e->chunk_len = chunk_len; e->prefix_len = prefix_len; e->target_ctas = target_ctas; e->pair_mode = pair_mode; e->fp8 = fp8;
        e->lens.assign(dec_ctx_lens, dec_ctx_lens + n_dec);
        layout_entry(*e);
        e->cur = 0;
        if (int rc = upload_plan(ctx, *e, 0, stream)) return rc;
        e->valid = true;
    }
    e->stamp = ++ctx->plan_clock;
    PlanBuffer& b = e->buf[e->cur];
    const Plan& plan = e->plan;

    // ---- q tensor maps (kept while the caller passes the same buffers); everything that can fail on the host happens
    // before the first enqueue on the caller's stream
    if (!fp8 && n_dec > 0 && !plan.items.empty())
        if (int rc = encode_q_map(&ctx->qd_map, q_dec, uint64_t(n_dec) * kHeads, 16)) return rc;
    if (chunk_len > 0 && plan.n_chunk_items > 0)
        if (int rc = encode_q_map(&ctx->qc_map, q_chunk, uint64_t(chunk_len) * kHeads, 64)) return rc;
    if (chunk_len > 0 && plan.n_pairs > 0)
        if (int rc = encode_q_map(&ctx->qp_map, q_chunk, uint64_t(chunk_len) * kHeads, 128)) return rc;

    if (b.upload_pending) {
        KAIROS_CUDA_TRY(cudaStreamWaitEvent(stream, b.uploaded, 0));
        if (cache_state == 2 && cudaEventQuery(b.uploaded) == cudaSuccess) b.upload_pending = false;
    }

    // ---- launch: a plan used again with the same buffers is replayed as a CUDA graph (one cudaGraphLaunch instead of 2-3
    // launches with their attributes); kairos_profile_enable forces direct launches because it brackets them with events
    bool graphed = false;
    if (ctx->use_graph && !ctx->profile) {
        if (b.exec && same_args(b.gargs, a)) {
            graphed = true;
        } else {
            if (b.same_args_uses > 0 && same_args(b.gargs, a)) {
                if (++b.same_args_uses >= 2) graphed = capture_graph(ctx, *e, b, a);
            } else {
                drop_graph(b);
                b.gargs = a;
                b.same_args_uses = 1;
            }
        }
    }
    if (graphed) {
        KAIROS_CUDA_TRY(cudaGraphLaunch(b.exec, stream));
    } else {
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (int rc = next_profile_events(ctx, &e0, &e1)) return rc;
        if (int rc = launch_step_kernels(ctx, *e, b, a, stream, e0, e1)) return rc;
    }
    KAIROS_CUDA_TRY(cudaEventRecord(b.last_use, stream));

    ctx->last_info[0] = int64_t(plan.items.size());
    ctx->last_info[1] = plan.n_decode_items;
    ctx->last_info[2] = plan.n_chunk_items + int64_t(plan.pair_items.size());
    ctx->last_info[3] = std::min<int64_t>(plan.n_pairs > 0 && plan.dec_ctas > 0 ? plan.dec_ctas : umma_resident_ctas(ctx), int64_t(plan.items.size()));
    ctx->last_info[4] = kernels_of(plan);
    ctx->last_info[5] = int64_t(kCounterBytes + size_t(plan.n_partial_slots) * kPartialSlotBytes);
    ctx->last_info[6] = plan.n_pairs;
    ctx->last_info[7] = cache_state;
    ctx->last_info[8] = graphed ? 1 : 0;
    ctx->last_info[9] = plan.dec_ctas;
    return KAIROS_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// a whole chunk schedule X = [chi(1) .. chi(m)] as m successive (append -> mixed step) steps
// ---------------------------------------------------------------------------------------------------------------
struct ScheduleArgs {
    int32_t n_dec;
    const void* q_dec;
    const int32_t* dec_page_tables;
    int32_t dec_table_stride;
    const void* dec_latent;
    const void* dec_k_rope;
    const void* q_prompt;
    const void* prompt_latent;
    const void* prompt_k_rope;
    const int32_t* prompt_page_table;
    int32_t prompt_table_len, prefix_len;
    void* out_dec;
    void* out_prompt;
    float* lse_dec;
    float* lse_prompt;
};

// Enqueues steps [0, m) on `stream` (the caller's, or the capture stream).  ev: 2 events per step (start, stop) or NULL.
static int enqueue_schedule(kairos_ctx* ctx, const ScheduleArgs& s, const std::vector<PlanEntry>& steps, const std::vector<int32_t>& lens0,
                            const int32_t* chunk_sizes, int32_t m, const uint8_t* arena, const std::vector<size_t>& plan_off,
                            size_t pos_off, cudaStream_t stream, cudaEvent_t* ev) {
    const bool grow = s.dec_latent != nullptr;
    int64_t done = 0;
    for (int32_t i = 0; i < m; ++i) {
        const int32_t C = chunk_sizes[i];
        const int32_t P = s.prefix_len + int32_t(done);
        if (ev) KAIROS_CUDA_TRY(cudaEventRecord(ev[2 * i], stream));
        if (grow && s.n_dec > 0)  // every in-flight decode caches its newest token first
            if (int rc = launch_append_decode(ctx, static_cast<const uint8_t*>(s.dec_latent) + size_t(i) * s.n_dec * kLatent * 2,
                                              static_cast<const uint8_t*>(s.dec_k_rope) + size_t(i) * s.n_dec * kRope * 2, s.n_dec,
                                              s.dec_page_tables, s.dec_table_stride,
                                              reinterpret_cast<const int32_t*>(arena + pos_off) + size_t(i) * s.n_dec, stream))
                return rc;
        if (C > 0)
            if (int rc = launch_append(ctx, static_cast<const uint8_t*>(s.prompt_latent) + size_t(done) * kLatent * 2,
                                       static_cast<const uint8_t*>(s.prompt_k_rope) + size_t(done) * kRope * 2, C, s.prompt_page_table, P, stream))
                return rc;
        StepArgs a{};
        a.n_dec = s.n_dec;
        a.q_dec = static_cast<const uint8_t*>(s.q_dec) + size_t(i) * s.n_dec * kHeads * kDim * 2;
        a.dec_page_tables = s.dec_page_tables;
        a.dec_table_stride = s.dec_table_stride;
        a.chunk_len = C;
        a.prefix_len = P;
        a.q_chunk = static_cast<const uint8_t*>(s.q_prompt) + size_t(done) * kHeads * kDim * 2;
        a.chunk_page_table = s.prompt_page_table;
        a.out_dec = static_cast<uint8_t*>(s.out_dec) + size_t(i) * s.n_dec * kHeads * kLatent * 2;
        a.out_chunk = static_cast<uint8_t*>(s.out_prompt) + size_t(done) * kHeads * kLatent * 2;
        a.lse_dec = s.lse_dec ? s.lse_dec + size_t(i) * s.n_dec * kHeads : nullptr;
        a.lse_chunk = s.lse_prompt ? s.lse_prompt + size_t(done) * kHeads : nullptr;
        const PlanEntry& e = steps[i];
        if (s.n_dec > 0 && !e.plan.items.empty())
            if (int rc = encode_q_map(&ctx->qd_map, a.q_dec, uint64_t(s.n_dec) * kHeads, 16)) return rc;
        if (C > 0 && e.plan.n_chunk_items > 0)
            if (int rc = encode_q_map(&ctx->qc_map, a.q_chunk, uint64_t(C) * kHeads, 64)) return rc;
        if (C > 0 && e.plan.n_pairs > 0)
            if (int rc = encode_q_map(&ctx->qp_map, a.q_chunk, uint64_t(C) * kHeads, 128)) return rc;
        PlanBuffer b;
        b.dev = const_cast<uint8_t*>(arena) + plan_off[i];
        cudaEvent_t pe0 = nullptr, pe1 = nullptr;  // kairos_profile_enable brackets each step's attention kernels (never while capturing)
        if (stream != ctx->capture_stream)
            if (int rc = next_profile_events(ctx, &pe0, &pe1)) return rc;
        if (int rc = launch_step_kernels(ctx, e, b, a, stream, pe0, pe1)) return rc;
        if (ev) KAIROS_CUDA_TRY(cudaEventRecord(ev[2 * i + 1], stream));
        done += C;
    }
    (void)lens0;
    return KAIROS_OK;
}

}  // namespace kairos

using namespace kairos;

extern "C" int kairos_run_schedule(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                                   int32_t dec_table_stride, const int32_t* dec_ctx_lens, const void* dec_latent,
                                   const void* dec_k_rope, int32_t prompt_len, const int32_t* chunk_sizes, int32_t n_steps,
                                   const void* q_prompt, const void* prompt_latent, const void* prompt_k_rope,
                                   const int32_t* prompt_page_table, int32_t prompt_table_len, int32_t prefix_len,
                                   void* out_dec, void* out_prompt, float* lse_dec, float* lse_prompt, double* step_us,
                                   double* ttft_us, void* cuda_stream) {
    if (!ctx) return fail(KAIROS_ERR_INVALID_ARG, "ctx is NULL");
    if (n_dec < 0 || prompt_len < 1 || n_steps < 1 || prefix_len < 0 || !chunk_sizes)
        return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: bad size or NULL chunk_sizes");
    if (!q_prompt || !prompt_latent || !prompt_k_rope || !prompt_page_table || !out_prompt)
        return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: NULL prompt argument");
    if (n_dec > 0 && (!q_dec || !dec_page_tables || !dec_ctx_lens || !out_dec || dec_table_stride < 1))
        return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: NULL decode argument");
    if ((dec_latent == nullptr) != (dec_k_rope == nullptr)) return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: dec_latent and dec_k_rope go together");
    int64_t total = 0;
    for (int32_t i = 0; i < n_steps; ++i) {
        if (chunk_sizes[i] < 1) return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: chunk_sizes[" + std::to_string(i) + "] < 1");
        total += chunk_sizes[i];
    }
    if (total != prompt_len) return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: chunk_sizes must sum to prompt_len");
    if (int64_t(prefix_len) + prompt_len > int64_t(prompt_table_len) * kPage)
        return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: prompt page table shorter than prefix_len + prompt_len");
    const bool grow = dec_latent != nullptr;
    for (int32_t j = 0; j < n_dec; ++j) {
        if (dec_ctx_lens[j] < (grow ? 0 : 1)) return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: dec_ctx_lens[" + std::to_string(j) + "] too small");
        if (int64_t(dec_ctx_lens[j]) + (grow ? n_steps : 0) > int64_t(dec_table_stride) * kPage)
            return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: decode " + std::to_string(j) + " outgrows its page table");
    }
    for (const void* ptr : {q_dec, q_prompt, prompt_latent, prompt_k_rope, dec_latent, dec_k_rope, static_cast<const void*>(out_dec),
                            static_cast<const void*>(out_prompt)})
        if (reinterpret_cast<uintptr_t>(ptr) % 16) return fail(KAIROS_ERR_INVALID_ARG, "run_schedule: device buffers must be 16-byte aligned");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    KAIROS_CUDA_TRY(cudaSetDevice(ctx->cfg.device));

    const ScheduleArgs s{n_dec, q_dec, dec_page_tables, dec_table_stride, dec_latent, dec_k_rope, q_prompt, prompt_latent, prompt_k_rope,
                         prompt_page_table, prompt_table_len, prefix_len, out_dec, out_prompt, lse_dec, lse_prompt};
    // ---- the cached schedule is replayed when every argument, length and chunk size is the same
    std::vector<uint8_t> key(sizeof(ScheduleArgs) + sizeof(int32_t) * (size_t(n_dec) + n_steps + 2));
    {
        uint8_t* k = key.data();
        std::memset(k, 0, key.size());
        ScheduleArgs z;
        std::memset(&z, 0, sizeof(z));  // padding bytes of the struct must compare equal
        z = s;
        std::memcpy(k, &z, sizeof(z)); k += sizeof(z);
        std::memcpy(k, &prompt_len, 4); k += 4;
        std::memcpy(k, &n_steps, 4); k += 4;
        if (n_dec) std::memcpy(k, dec_ctx_lens, sizeof(int32_t) * size_t(n_dec));
        k += sizeof(int32_t) * size_t(n_dec);
        std::memcpy(k, chunk_sizes, sizeof(int32_t) * size_t(n_steps));
    }
    ScheduleCache& sc = ctx->schedule;
    const bool want_steps = step_us != nullptr || ctx->profile;  // both launch the steps one by one (event brackets)
    const bool planned = !sc.key.empty() && sc.key == key;  // plans of every step are in the arena already
    if (!planned) {
        // ---- plan every step (a0) and pack the work lists and the decodes' append positions into one arena
        if (sc.exec) { cudaGraphExecDestroy(sc.exec); sc.exec = nullptr; }
        sc.key.clear();
        sc.steps.assign(size_t(n_steps), PlanEntry());
        sc.plan_off.assign(size_t(n_steps), 0);
        std::vector<int32_t> lens(dec_ctx_lens, dec_ctx_lens + n_dec);
        size_t off = 0, ws_needed = 0;
        int64_t done = 0;
        sc.kernels = 0;
        for (int32_t i = 0; i < n_steps; ++i) {
            if (grow) for (int32_t j = 0; j < n_dec; ++j) lens[j] = dec_ctx_lens[j] + i + 1;
            PlanEntry& e = sc.steps[i];
            build_plan(lens.data(), n_dec, chunk_sizes[i], prefix_len + int32_t(done), umma_resident_ctas(ctx), umma_chunk_tile_tokens(),
                       &e.plan, pair_mode_for(ctx, lens.data(), n_dec, chunk_sizes[i], prefix_len + int32_t(done)), pair_tile_tokens());
            layout_entry(e);
            sc.plan_off[i] = off;
            off += (e.total_bytes + 255) / 256 * 256;
            ws_needed = std::max(ws_needed, kCounterBytes + size_t(e.plan.n_partial_slots) * kPartialSlotBytes);
            sc.kernels += kernels_of(e.plan) + 1 + (grow && n_dec > 0 ? 1 : 0);
            done += chunk_sizes[i];
        }
        if (ws_needed > ctx->cfg.workspace_bytes)
            return fail(KAIROS_ERR_WORKSPACE, "run_schedule: workspace too small: need " + std::to_string(ws_needed) + " bytes");
        sc.pos_off = off;
        off += (size_t(n_steps) * std::max(n_dec, 1) * 4 + 255) / 256 * 256;
        KAIROS_CUDA_TRY(cudaStreamSynchronize(stream));  // a previous schedule may still be reading the arena
        if (sc.cap < off) {
            if (sc.host) cudaFreeHost(sc.host);
            if (sc.dev) cudaFree(sc.dev);
            sc.host = sc.dev = nullptr;
            sc.cap = 0;
            KAIROS_CUDA_TRY(cudaMallocHost(&sc.host, off));
            KAIROS_CUDA_TRY(cudaMalloc(&sc.dev, off));
            sc.cap = off;
        }
        uint8_t* h = static_cast<uint8_t*>(sc.host);
        for (int32_t i = 0; i < n_steps; ++i) {
            const PlanEntry& e = sc.steps[i];
            uint8_t* hp = h + sc.plan_off[i];
            std::memcpy(hp, e.plan.items.data(), e.items_bytes);
            if (e.comb_bytes) std::memcpy(hp + e.comb_off, e.plan.combines.data(), e.comb_bytes);
            if (e.pair_bytes) std::memcpy(hp + e.pair_off, e.plan.pair_items.data(), e.pair_bytes);
        }
        int32_t* pos = reinterpret_cast<int32_t*>(h + sc.pos_off);
        for (int32_t i = 0; i < n_steps; ++i)
            for (int32_t j = 0; j < n_dec; ++j) pos[size_t(i) * n_dec + j] = dec_ctx_lens[j] + i;  // the slot of step i's new token
        KAIROS_CUDA_TRY(cudaMemcpyAsync(sc.dev, sc.host, off, cudaMemcpyHostToDevice, stream));
        sc.key = key;
    }
    {
        // ---- one CUDA graph for the whole schedule (programmatic launch edges kept), captured on first use without timing brackets
        std::vector<int32_t> lens(dec_ctx_lens, dec_ctx_lens + n_dec);
        if (!sc.exec && ctx->use_graph && !want_steps && ctx->capture_stream &&
            cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const int rc = enqueue_schedule(ctx, s, sc.steps, lens, chunk_sizes, n_steps, static_cast<const uint8_t*>(sc.dev), sc.plan_off,
                                            sc.pos_off, ctx->capture_stream, nullptr);
            cudaGraph_t graph = nullptr;
            const cudaError_t ce = cudaStreamEndCapture(ctx->capture_stream, &graph);
            bool ok = rc == KAIROS_OK && ce == cudaSuccess && graph != nullptr;
            if (ok) ok = cudaGraphInstantiate(&sc.exec, graph, 0) == cudaSuccess;
            if (graph) cudaGraphDestroy(graph);
            if (!ok) {  // not an error of the schedule: graphs are switched off for this context, the steps are launched one by one
                cudaGetLastError();
                sc.exec = nullptr;
                ctx->use_graph = 0;
            }
        }
    }
    // ---- run it: TTFT_dec (Eq. 6's left-hand side, measured) is the device time from the first append to the last kernel
    const bool timed = ttft_us || step_us;
    std::vector<cudaEvent_t> ev;
    struct EvGuard {
        std::vector<cudaEvent_t>& v;
        ~EvGuard() { for (auto e : v) cudaEventDestroy(e); }
    } guard{ev};
    const int n_ev = timed ? 2 + (step_us ? 2 * n_steps : 0) : 0;
    for (int i = 0; i < n_ev; ++i) {
        cudaEvent_t e;
        KAIROS_CUDA_TRY(cudaEventCreate(&e));
        ev.push_back(e);
    }
    if (timed) KAIROS_CUDA_TRY(cudaEventRecord(ev[0], stream));
    if (sc.exec && !want_steps) {
        KAIROS_CUDA_TRY(cudaGraphLaunch(sc.exec, stream));
    } else {
        std::vector<int32_t> lens(dec_ctx_lens, dec_ctx_lens + n_dec);
        if (int rc = enqueue_schedule(ctx, s, sc.steps, lens, chunk_sizes, n_steps, static_cast<const uint8_t*>(sc.dev), sc.plan_off,
                                      sc.pos_off, stream, step_us ? ev.data() + 2 : nullptr))
            return rc;
    }
    {   // kairos_last_plan_info: the LAST step's plan; [4] counts every kernel of the schedule (appends included)
        const Plan& lp = sc.steps.back().plan;
        std::memset(ctx->last_info, 0, sizeof(ctx->last_info));
        ctx->last_info[0] = int64_t(lp.items.size());
        ctx->last_info[1] = lp.n_decode_items;
        ctx->last_info[2] = lp.n_chunk_items + int64_t(lp.pair_items.size());
        ctx->last_info[3] = std::min<int64_t>(lp.n_pairs > 0 && lp.dec_ctas > 0 ? lp.dec_ctas : umma_resident_ctas(ctx), int64_t(lp.items.size()));
        ctx->last_info[4] = sc.kernels;
        ctx->last_info[5] = int64_t(kCounterBytes + size_t(lp.n_partial_slots) * kPartialSlotBytes);
        ctx->last_info[6] = lp.n_pairs;
        ctx->last_info[7] = planned ? 2 : 0;
        ctx->last_info[8] = (sc.exec && !want_steps) ? 1 : 0;
        ctx->last_info[9] = lp.dec_ctas;
    }
    if (timed) {
        KAIROS_CUDA_TRY(cudaEventRecord(ev[1], stream));
        KAIROS_CUDA_TRY(cudaEventSynchronize(ev[1]));
        float ms = 0.f;
        KAIROS_CUDA_TRY(cudaEventElapsedTime(&ms, ev[0], ev[1]));
        if (ttft_us) *ttft_us = double(ms) * 1e3;
        for (int32_t i = 0; step_us && i < n_steps; ++i) {
            KAIROS_CUDA_TRY(cudaEventElapsedTime(&ms, ev[2 + 2 * i], ev[3 + 2 * i]));
            step_us[i] = double(ms) * 1e3;
        }
    }
    return KAIROS_OK;
}

namespace kairos {
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
    if (cfg->workspace_bytes < kCounterBytes)
        return fail(KAIROS_ERR_WORKSPACE, "workspace must hold at least 256 bytes (work-queue counters)");
    kairos_ctx* ctx = new (std::nothrow) kairos_ctx();
    if (!ctx) return fail(KAIROS_ERR_INVALID_ARG, "out of host memory");
    ctx->cfg = *cfg;
    ctx->sm_count = prop.multiProcessorCount;
    int rc = umma_init(ctx);
    if (rc == KAIROS_OK) rc = pair_init(ctx);
    if (rc == KAIROS_OK && cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) != cudaSuccess)
        rc = fail(KAIROS_ERR_CUDA, "cudaStreamCreateWithFlags(copy stream) failed");
    if (rc == KAIROS_OK && cudaStreamCreateWithFlags(&ctx->capture_stream, cudaStreamNonBlocking) != cudaSuccess)
        rc = fail(KAIROS_ERR_CUDA, "cudaStreamCreateWithFlags(capture stream) failed");
    if (rc != KAIROS_OK) {
        const std::string msg = g_last_error;
        kairos_destroy(ctx);
        g_last_error = msg;
        return rc;
    }
    *out = ctx;
    return KAIROS_OK;
}

int kairos_destroy(kairos_ctx* ctx) {
    if (!ctx) return KAIROS_OK;
    cudaSetDevice(ctx->cfg.device);
    for (PlanEntry& e : ctx->plans)
        for (PlanBuffer& b : e.buf) {
            if (b.ever_used && b.uploaded) cudaEventSynchronize(b.uploaded);
            if (b.ever_used && b.last_use) cudaEventSynchronize(b.last_use);
            if (b.exec) cudaGraphExecDestroy(b.exec);
            if (b.host) cudaFreeHost(b.host);
            if (b.dev) cudaFree(b.dev);
            if (b.uploaded) cudaEventDestroy(b.uploaded);
            if (b.last_use) cudaEventDestroy(b.last_use);
        }
    if (ctx->host_stage.dev) cudaFree(ctx->host_stage.dev);
    for (auto e : ctx->host_stage.events) cudaEventDestroy(e);
    if (ctx->host_stage.in) cudaStreamDestroy(ctx->host_stage.in);
    if (ctx->host_stage.out) cudaStreamDestroy(ctx->host_stage.out);
    if (ctx->schedule.exec) cudaGraphExecDestroy(ctx->schedule.exec);
    if (ctx->schedule.host) cudaFreeHost(ctx->schedule.host);
    if (ctx->schedule.dev) cudaFree(ctx->schedule.dev);
    if (ctx->table_buf) cudaFree(ctx->table_buf);
    if (ctx->flush_buf) cudaFree(ctx->flush_buf);
    for (auto e : ctx->prof_events) cudaEventDestroy(e);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->capture_stream) cudaStreamDestroy(ctx->capture_stream);
    delete ctx;
    return KAIROS_OK;
}

int kairos_tune_step(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                     const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len, const void* q_chunk,
                     const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec, void* out_chunk, int32_t reps,
                     int32_t* chosen_mode, double* chosen_us, double* default_us, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (reps < 1) return fail(KAIROS_ERR_INVALID_ARG, "tune: reps < 1");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (chosen_mode) *chosen_mode = -1;
    if (chunk_len <= 0 || n_dec <= 0) {  // one grid only: nothing to order
        if (chosen_us) *chosen_us = 0.0;
        if (default_us) *default_us = 0.0;
        return KAIROS_OK;
    }
    const int32_t tiles = (chunk_len + pair_tile_tokens() - 1) / pair_tile_tokens();
    const int32_t max_pairs = std::min(tiles, ctx->sm_count / 2);
    // candidates: the planner's own choice first, then every cluster first, a few clusters first, decode grid first beside n clusters
    std::vector<int32_t> modes{-1, -(max_pairs + 1)};
    for (int32_t n : {8, 16, 24, 32, 48})
        if (n < max_pairs) modes.push_back(-(n + 1));
    for (int32_t n : {20, 28, 36, 44, 52, 60})
        if (n < max_pairs && ctx->sm_count - 2 * n >= 2) modes.push_back(n);
    if (tiles <= 64) modes.push_back(0);
    const uint64_t key = shape_key(dec_ctx_lens, n_dec, chunk_len, prefix_len);
    for (size_t i = 0; i < ctx->tuned.size(); ++i)
        if (ctx->tuned[i].key == key) { ctx->tuned.erase(ctx->tuned.begin() + long(i)); break; }
    const int saved_force = ctx->force_pairs, saved_graph = ctx->use_graph;
    ctx->use_graph = 0;  // candidates are timed as direct launches: the order of the grids is what differs
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = KAIROS_OK;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = fail(KAIROS_ERR_CUDA, "tune: cudaEventCreate failed");
    double best = 0.0, def = 0.0;
    int32_t best_mode = -1;
    std::vector<double> ts;
    for (size_t m = 0; m < modes.size() && rc == KAIROS_OK; ++m) {
        ctx->force_pairs = modes[m];
        ts.clear();
        for (int32_t it = 0; it < 2 + reps && rc == KAIROS_OK; ++it) {
            if (cudaEventRecord(e0, stream) != cudaSuccess) { rc = fail(KAIROS_ERR_CUDA, "tune: cudaEventRecord failed"); break; }
            rc = mixed_step_impl(ctx, n_dec, q_dec, dec_page_tables, dec_table_stride, dec_ctx_lens, chunk_len, prefix_len, q_chunk,
                                 chunk_page_table, chunk_table_len, out_dec, out_chunk, nullptr, nullptr, stream);
            if (rc != KAIROS_OK) break;
            if (cudaEventRecord(e1, stream) != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) { rc = fail(KAIROS_ERR_CUDA, "tune: step failed on the device"); break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (it >= 2) ts.push_back(double(ms) * 1e3);
        }
        if (rc != KAIROS_OK) break;
        std::sort(ts.begin(), ts.end());
        const double med = ts[ts.size() / 2];
        if (m == 0) def = med;
        if (m == 0 || med < best) { best = med; best_mode = modes[m]; }
    }
    ctx->force_pairs = saved_force;
    ctx->use_graph = saved_graph;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (rc != KAIROS_OK) return rc;
    if (best_mode != -1 && best < 0.97 * def) {  // pinned only when it beats the planner's own order by more than the noise
        if (ctx->tuned.size() >= 256) ctx->tuned.erase(ctx->tuned.begin());
        ctx->tuned.push_back(TunedShape{key, best_mode});
    } else {
        best_mode = -1;
        best = def;
    }
    for (PlanEntry& e : ctx->plans) {  // plans of this shape were built under forced orders: drop them
        for (PlanBuffer& b : e.buf) drop_graph(b);
        e.valid = false;
    }
    ctx->schedule.key.clear();
    if (chosen_mode) *chosen_mode = best_mode;
    if (chosen_us) *chosen_us = best;
    if (default_us) *default_us = def;
    return KAIROS_OK;
}

int kairos_debug_set(kairos_ctx* ctx, const char* key, int32_t value) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!key) return fail(KAIROS_ERR_INVALID_ARG, "key is NULL");
    const std::string k(key);
    if (k == "pairs") ctx->force_pairs = value;
    else if (k == "dec_only") ctx->force_dec_only = value;
    else if (k == "copy_stream") ctx->use_copy_stream = value != 0;
    else if (k == "graph") ctx->use_graph = value != 0;
    else if (k == "plan_cache") ctx->use_plan_cache = value != 0;
    else if (k == "host_slice_tokens") ctx->host_slice_tokens = value;
    else return fail(KAIROS_ERR_INVALID_ARG, "unknown debug key '" + k + "'");
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

int kairos_absorb_q(kairos_ctx* ctx, const void* q_nope, const void* q_rope, const void* w_uk_t, int32_t n, void* q_out,
                    void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n < 0) return fail(KAIROS_ERR_INVALID_ARG, "n < 0");
    if (n == 0) return KAIROS_OK;
    if (!q_nope || !q_rope || !w_uk_t || !q_out) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    for (const void* p : {q_nope, q_rope, w_uk_t, static_cast<const void*>(q_out)})
        if (reinterpret_cast<uintptr_t>(p) % 16) return fail(KAIROS_ERR_INVALID_ARG, "buffers must be 16-byte aligned");
    return launch_absorb_q(ctx, q_nope, q_rope, w_uk_t, n, q_out, static_cast<cudaStream_t>(cuda_stream));
}

int kairos_project_out(kairos_ctx* ctx, const void* o_lat, const void* w_uv_t, int32_t n, void* v_out, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n < 0) return fail(KAIROS_ERR_INVALID_ARG, "n < 0");
    if (n == 0) return KAIROS_OK;
    if (!o_lat || !w_uv_t || !v_out) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    for (const void* p : {o_lat, w_uv_t, static_cast<const void*>(v_out)})
        if (reinterpret_cast<uintptr_t>(p) % 16) return fail(KAIROS_ERR_INVALID_ARG, "buffers must be 16-byte aligned");
    return launch_project_out(ctx, o_lat, w_uv_t, n, v_out, static_cast<cudaStream_t>(cuda_stream));
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

// ---- the fp8 latent cache ------------------------------------------------------------------------------
int kairos_fp8_attach(kairos_ctx* ctx, void* pool8, int32_t num_pages) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!pool8 || num_pages < 1) return fail(KAIROS_ERR_INVALID_ARG, "NULL pool8 or num_pages < 1");
    if (reinterpret_cast<uintptr_t>(pool8) % 128) return fail(KAIROS_ERR_INVALID_ARG, "pool8 must be 128-byte aligned");
    return fp8_attach(ctx, pool8, num_pages);
}

int kairos_fp8_append(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens, const int32_t* page_table,
                      int32_t table_len, int32_t start_pos, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!ctx->fp8.attached) return fail(KAIROS_ERR_INVALID_ARG, "no fp8 pool attached (kairos_fp8_attach)");
    if (n_tokens < 0 || start_pos < 0 || table_len < 0) return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    if (n_tokens == 0) return KAIROS_OK;
    if (!latent || !k_rope || !page_table) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    if (int64_t(start_pos) + n_tokens > int64_t(table_len) * kPage)
        return fail(KAIROS_ERR_INVALID_ARG, "start_pos + n_tokens beyond table_len*64");
    if (reinterpret_cast<uintptr_t>(latent) % 16 || reinterpret_cast<uintptr_t>(k_rope) % 16)
        return fail(KAIROS_ERR_INVALID_ARG, "latent / k_rope must be 16-byte aligned");
    return launch_fp8_append(ctx, latent, k_rope, n_tokens, page_table, start_pos, static_cast<cudaStream_t>(cuda_stream));
}

int kairos_fp8_append_decode_tokens(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n, const int32_t* page_tables,
                                    int32_t table_stride, const int32_t* positions, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!ctx->fp8.attached) return fail(KAIROS_ERR_INVALID_ARG, "no fp8 pool attached (kairos_fp8_attach)");
    if (n < 0 || table_stride < 1) return fail(KAIROS_ERR_INVALID_ARG, "n < 0 or table_stride < 1");
    if (n == 0) return KAIROS_OK;
    if (!latent || !k_rope || !page_tables || !positions) return fail(KAIROS_ERR_INVALID_ARG, "NULL pointer");
    if (reinterpret_cast<uintptr_t>(latent) % 16 || reinterpret_cast<uintptr_t>(k_rope) % 16)
        return fail(KAIROS_ERR_INVALID_ARG, "latent / k_rope must be 16-byte aligned");
    return launch_fp8_append_decode(ctx, latent, k_rope, n, page_tables, table_stride, positions, static_cast<cudaStream_t>(cuda_stream));
}

int kairos_fp8_mixed_step(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                          const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len, const void* q_chunk,
                          const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec, void* out_chunk, float* lse_dec,
                          float* lse_chunk, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!ctx->fp8.attached) return fail(KAIROS_ERR_INVALID_ARG, "no fp8 pool attached (kairos_fp8_attach)");
    return mixed_step_impl(ctx, n_dec, q_dec, dec_page_tables, dec_table_stride, dec_ctx_lens, chunk_len, prefix_len, q_chunk,
                           chunk_page_table, chunk_table_len, out_dec, out_chunk, lse_dec, lse_chunk, static_cast<cudaStream_t>(cuda_stream),
                           /*fp8=*/1);
}

int kairos_fp8_decode(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                      int32_t dec_table_stride, const int32_t* dec_ctx_lens, void* out_dec, float* lse_dec, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (!ctx->fp8.attached) return fail(KAIROS_ERR_INVALID_ARG, "no fp8 pool attached (kairos_fp8_attach)");
    return mixed_step_impl(ctx, n_dec, q_dec, dec_page_tables, dec_table_stride, dec_ctx_lens, 0, 0, nullptr, nullptr, 0, out_dec,
                           nullptr, lse_dec, nullptr, static_cast<cudaStream_t>(cuda_stream), /*fp8=*/1);
}

// ---- decode attention for callers that may not allocate (scratch = a fixed __device__ array in attn_umma.cu) ------------------
int kairos_decode_static(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                         const int32_t* dec_ctx_lens, void* out_dec, float* lse_dec, void* cuda_stream) {
    if (int rc = check_ctx(ctx)) return rc;
    if (n_dec < 0) return fail(KAIROS_ERR_INVALID_ARG, "negative size");
    if (n_dec == 0) return KAIROS_OK;
    if (!q_dec || !dec_page_tables || !dec_ctx_lens || !out_dec) return fail(KAIROS_ERR_INVALID_ARG, "NULL decode argument");
    if (dec_table_stride < 1) return fail(KAIROS_ERR_INVALID_ARG, "dec_table_stride < 1");
    if (reinterpret_cast<uintptr_t>(q_dec) % 16 || reinterpret_cast<uintptr_t>(out_dec) % 16 || reinterpret_cast<uintptr_t>(lse_dec) % 4)
        return fail(KAIROS_ERR_INVALID_ARG, "q_dec / out_dec must be 16-byte aligned (lse_dec: 4)");
    if (n_dec > KAIROS_STATIC_MAX_DECODES)
        return fail(KAIROS_ERR_WORKSPACE, "kairos_decode_static takes at most " + std::to_string(KAIROS_STATIC_MAX_DECODES) +
                                              " decodes per call (got " + std::to_string(n_dec) + "): its scratch is a fixed array");
    for (int32_t i = 0; i < n_dec; ++i) {
        if (dec_ctx_lens[i] < 1) return fail(KAIROS_ERR_INVALID_ARG, "dec_ctx_lens[" + std::to_string(i) + "] < 1");
        if (int64_t(dec_ctx_lens[i]) > int64_t(dec_table_stride) * kPage)
            return fail(KAIROS_ERR_INVALID_ARG, "dec_ctx_lens[" + std::to_string(i) + "] beyond its page table");
    }
    return launch_decode_static(ctx, n_dec, q_dec, dec_page_tables, dec_table_stride, dec_ctx_lens, out_dec, lse_dec,
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
    // ---- slices.  A large chunk is cut into slices of whole rounds of the cluster grid (sm_count / 2 tiles of 8 tokens) and
    // the slices run as successive mixed steps over a growing prefix -- the same tiles over the same keys, so by chunk
    // invariance the same rows -- while the next slice's queries come up on a second stream and the previous
    // slice's outputs go down on a third: the copies (34.8 KB per chunk token over PCIe) hide behind the attention instead
    // of bracketing it.  At most 7 slices (+ the decodes' own step), so that their plans stay in the context's cache from call to call.
    const int32_t tile = pair_tile_tokens();
    const int32_t round_tokens = (ctx->sm_count / 2) * tile;
    int32_t slice = chunk_len;
    if (ctx->host_slice_tokens > 0) slice = (ctx->host_slice_tokens + tile - 1) / tile * tile;
    else if (chunk_len >= 2 * round_tokens) slice = (chunk_len + 7 * round_tokens - 1) / (7 * round_tokens) * round_tokens;
    const int32_t n_slices = chunk_len > 0 ? (chunk_len + slice - 1) / slice : 1;
    HostStage& hs = ctx->host_stage;
    cudaStream_t s_in = stream, s_out = stream;
    if (n_slices > 1) {
        if (!hs.in) KAIROS_CUDA_TRY(cudaStreamCreateWithFlags(&hs.in, cudaStreamNonBlocking));
        if (!hs.out) KAIROS_CUDA_TRY(cudaStreamCreateWithFlags(&hs.out, cudaStreamNonBlocking));
        while (hs.events.size() < size_t(2 * n_slices + 2)) {
            cudaEvent_t e;
            KAIROS_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            hs.events.push_back(e);
        }
        s_in = hs.in;
        s_out = hs.out;
    }
    uint64_t h2d = 0, d2h = 0;
    auto up = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!bytes) return cudaSuccess;
        h2d += bytes;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, s_in);
    };
    auto down = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!bytes || !dst) return cudaSuccess;
        d2h += bytes;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s_out);
    };
    // In a sliced step the decodes run first as a step of their own: they need only q_dec and the page tables (a few hundred
    // KB), so their attention covers the upload of the first slice's queries.
    const bool dec_first = n_slices > 1 && n_dec > 0;
    auto run = [&]() -> int {
        KAIROS_CUDA_TRY(up(d_qd, q_dec, size_t(n_dec) * kHeads * kDim * 2));
        KAIROS_CUDA_TRY(up(d_dpt, dec_page_tables, size_t(n_dec) * dec_table_stride * 4));
        if (dec_first) {
            cudaEvent_t e_in = hs.events[2 * n_slices], e_done = hs.events[2 * n_slices + 1];
            KAIROS_CUDA_TRY(cudaEventRecord(e_in, s_in));
            KAIROS_CUDA_TRY(cudaStreamWaitEvent(stream, e_in, 0));
            if (int rc = mixed_step_impl(ctx, n_dec, d_qd, reinterpret_cast<const int32_t*>(d_dpt), dec_table_stride, dec_ctx_lens, 0, 0,
                                         nullptr, nullptr, 0, d_od, nullptr, lse_dec ? reinterpret_cast<float*>(d_ld) : nullptr, nullptr,
                                         stream))
                return rc;
            KAIROS_CUDA_TRY(cudaEventRecord(e_done, stream));
            KAIROS_CUDA_TRY(cudaStreamWaitEvent(s_out, e_done, 0));
            KAIROS_CUDA_TRY(down(out_dec, d_od, size_t(n_dec) * kHeads * kLatent * 2));
            KAIROS_CUDA_TRY(down(lse_dec, d_ld, size_t(n_dec) * kHeads * 4));
        }
        KAIROS_CUDA_TRY(up(d_cpt, chunk_page_table, size_t(chunk_len > 0 ? chunk_table_len : 0) * 4));
        KAIROS_CUDA_TRY(up(d_lat, chunk_latent, size_t(chunk_len) * kLatent * 2));
        KAIROS_CUDA_TRY(up(d_rope, chunk_k_rope, size_t(chunk_len) * kRope * 2));
        for (int32_t i = 0; i < n_slices; ++i) {  // every slice's queries, in order, behind the small inputs
            const int32_t off = i * slice, len = std::min(slice, chunk_len - off);
            KAIROS_CUDA_TRY(up(d_qc + size_t(off) * kHeads * kDim * 2, static_cast<const uint8_t*>(q_chunk) + size_t(off) * kHeads * kDim * 2,
                               size_t(len) * kHeads * kDim * 2));
            if (n_slices > 1) KAIROS_CUDA_TRY(cudaEventRecord(hs.events[2 * i], s_in));
        }
        for (int32_t i = 0; i < n_slices; ++i) {
            const int32_t off = i * slice, len = std::min(slice, chunk_len - off);
            if (n_slices > 1) KAIROS_CUDA_TRY(cudaStreamWaitEvent(stream, hs.events[2 * i], 0));
            if (i == 0 && chunk_len > 0) {  // the whole chunk is appended once: a slice's rows see no key past their own position
                if (int rc = kairos_append_latent(ctx, d_lat, d_rope, chunk_len, reinterpret_cast<const int32_t*>(d_cpt),
                                                  chunk_table_len, prefix_len, cuda_stream))
                    return rc;
            }
            const int32_t nd = (i == 0 && !dec_first) ? n_dec : 0;
            if (int rc = mixed_step_impl(ctx, nd, d_qd, reinterpret_cast<const int32_t*>(d_dpt), dec_table_stride, dec_ctx_lens, len,
                                         prefix_len + off, d_qc + size_t(off) * kHeads * kDim * 2, reinterpret_cast<const int32_t*>(d_cpt),
                                         chunk_table_len, d_od, d_oc + size_t(off) * kHeads * kLatent * 2,
                                         lse_dec ? reinterpret_cast<float*>(d_ld) : nullptr,
                                         lse_chunk ? reinterpret_cast<float*>(d_lc) + size_t(off) * kHeads : nullptr, stream))
                return rc;
            if (n_slices > 1) {
                KAIROS_CUDA_TRY(cudaEventRecord(hs.events[2 * i + 1], stream));
                KAIROS_CUDA_TRY(cudaStreamWaitEvent(s_out, hs.events[2 * i + 1], 0));
            }
            if (i == 0 && !dec_first) {
                KAIROS_CUDA_TRY(down(out_dec, d_od, size_t(n_dec) * kHeads * kLatent * 2));
                KAIROS_CUDA_TRY(down(lse_dec, d_ld, size_t(n_dec) * kHeads * 4));
            }
            KAIROS_CUDA_TRY(down(out_chunk ? static_cast<uint8_t*>(out_chunk) + size_t(off) * kHeads * kLatent * 2 : nullptr,
                                 d_oc + size_t(off) * kHeads * kLatent * 2, size_t(len) * kHeads * kLatent * 2));
            KAIROS_CUDA_TRY(down(lse_chunk ? lse_chunk + size_t(off) * kHeads : nullptr, d_lc + size_t(off) * kHeads * 4,
                                 size_t(len) * kHeads * 4));
        }
        return KAIROS_OK;
    };
    const int rc = run();
    // nothing of this call is left in flight when it returns, whether it succeeded or not (the host buffers are the caller's)
    cudaError_t e1 = cudaSuccess, e2 = cudaSuccess, e3 = cudaStreamSynchronize(stream);
    if (n_slices > 1) {
        e1 = cudaStreamSynchronize(s_in);
        e2 = cudaStreamSynchronize(s_out);
    }
    if (rc) return rc;
    KAIROS_CUDA_TRY(e3);
    KAIROS_CUDA_TRY(e1);
    KAIROS_CUDA_TRY(e2);
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
    for (int32_t i = 0; i < n && i < 10; ++i) info[i] = ctx->last_info[i];
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

const char* kairos_version(void) {
    return "kairos-b200 sm_100a r2 (tcgen05 split-KV decode grid + 2-CTA chunk clusters, time-shared persistent grids, cached plans replayed as CUDA graphs)";
}

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
    // every point must fit the pool (the largest B and the largest K need not occur together)
    int64_t need_pages = 0;
    for (int iB = 0; iB < nB; ++iB)
        for (int iK = 0; iK < nK; ++iK)
            need_pages = std::max(need_pages, int64_t(Bs[iB]) * ((Ks[iK] + kPage - 1) / kPage));
    const int64_t max_chunk_pages = maxC > 0 ? (int64_t(prefix_len) + maxC + kPage - 1) / kPage : 0;
    if (need_pages + max_chunk_pages > ctx->cfg.num_pages)
        return fail(KAIROS_ERR_WORKSPACE, "pool has too few pages for the largest grid point: need " +
                                              std::to_string(need_pages + max_chunk_pages));
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    KAIROS_CUDA_TRY(cudaSetDevice(ctx->cfg.device));
    const int32_t stride = std::max(1, (maxK + kPage - 1) / kPage);
    // one scratch allocation kept by the context (grown on demand): q_dec | q_chunk | out_dec | out_chunk | page tables
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    const size_t nqd = size_t(std::max(maxB, 1)) * kHeads * kDim, nqc = size_t(std::max(maxC, 1)) * kHeads * kDim;
    const size_t b_qd = al(nqd * 2), b_qc = al(nqc * 2);
    const size_t b_od = al(size_t(std::max(maxB, 1)) * kHeads * kLatent * 2), b_oc = al(size_t(std::max(maxC, 1)) * kHeads * kLatent * 2);
    const size_t b_dpt = al(size_t(std::max(maxB, 1)) * stride * 4), b_cpt = al(size_t(std::max<int64_t>(max_chunk_pages, 1)) * 4);
    const size_t total = b_qd + b_qc + b_od + b_oc + b_dpt + b_cpt;
    if (ctx->table_bytes < total) {
        KAIROS_CUDA_TRY(cudaStreamSynchronize(stream));
        if (ctx->table_buf) cudaFree(ctx->table_buf);
        ctx->table_buf = nullptr;
        ctx->table_bytes = 0;
        KAIROS_CUDA_TRY(cudaMalloc(&ctx->table_buf, total));
        ctx->table_bytes = total;
    }
    const size_t flush_bytes = size_t(256) << 20;  // > 126 MB L2
    if (flush_l2 && !ctx->flush_buf) KAIROS_CUDA_TRY(cudaMalloc(&ctx->flush_buf, flush_bytes));
    uint8_t* p = static_cast<uint8_t*>(ctx->table_buf);
    uint16_t* q_dec = reinterpret_cast<uint16_t*>(p);    p += b_qd;
    uint16_t* q_chunk = reinterpret_cast<uint16_t*>(p);  p += b_qc;
    void* o_dec = p;                                     p += b_od;
    void* o_chunk = p;                                   p += b_oc;
    int32_t* dpt = reinterpret_cast<int32_t*>(p);        p += b_dpt;
    int32_t* cpt = reinterpret_cast<int32_t*>(p);
    fill_q_kernel<<<256, 256, 0, stream>>>(q_dec, nqd, 0x1234u);
    fill_q_kernel<<<256, 256, 0, stream>>>(q_chunk, nqc, 0x9876u);
    KAIROS_CUDA_TRY(cudaGetLastError());
    // one event pair per timed rep: the reps of a point are enqueued back to back (the host runs ahead while the flush
    // kernel or the previous step executes), so an interval is the device time of the step, not the host's enqueue time
    struct Events {
        std::vector<cudaEvent_t> ev;
        ~Events() { for (auto e : ev) cudaEventDestroy(e); }
    } events;
    for (int i = 0; i < 2 * reps; ++i) {
        cudaEvent_t e;
        KAIROS_CUDA_TRY(cudaEventCreate(&e));
        events.ev.push_back(e);
    }
    std::vector<int32_t> h_dpt, h_cpt, lens;
    std::vector<double> times;
    for (int iB = 0; iB < nB; ++iB)
        for (int iK = 0; iK < nK; ++iK)
            for (int iC = 0; iC < nC; ++iC) {
                const int32_t B = Bs[iB], K = Ks[iK], C = Cs[iC];
                const size_t o = (size_t(iB) * nK + iK) * nC + iC;
                if (B == 0 && C == 0) { out_median_us[o] = 0.0; if (out_min_us) out_min_us[o] = 0.0; continue; }
                // distinct pages, strided through the pool (a step coprime with num_pages visits each page once)
                const int64_t kp = (K + kPage - 1) / kPage, cp = C > 0 ? (int64_t(prefix_len) + C + kPage - 1) / kPage : 0;
                const int64_t np = ctx->cfg.num_pages;
                int64_t step = (np / 2) | 1;
                while (std::gcd(step, np) != 1) step += 2;
                auto page_of = [&](int64_t i) { return int32_t((i * step) % np); };
                h_dpt.assign(size_t(std::max(B, 1)) * stride, 0);
                for (int64_t b = 0; b < B; ++b)
                    for (int64_t pg = 0; pg < kp; ++pg) h_dpt[size_t(b) * stride + pg] = page_of(b * kp + pg);
                h_cpt.assign(size_t(std::max<int64_t>(cp, 1)), 0);
                for (int64_t pg = 0; pg < cp; ++pg) h_cpt[size_t(pg)] = page_of(int64_t(B) * kp + pg);
                lens.assign(size_t(std::max(B, 1)), K);
                KAIROS_CUDA_TRY(cudaMemcpyAsync(dpt, h_dpt.data(), h_dpt.size() * 4, cudaMemcpyHostToDevice, stream));
                KAIROS_CUDA_TRY(cudaMemcpyAsync(cpt, h_cpt.data(), h_cpt.size() * 4, cudaMemcpyHostToDevice, stream));
                KAIROS_CUDA_TRY(cudaStreamSynchronize(stream));  // the pageable sources above are reused by the next point
                for (int it = 0; it < warmup + reps; ++it) {
                    if (flush_l2) {
                        flush_kernel<<<1184, 256, 0, stream>>>(static_cast<uint4*>(ctx->flush_buf), flush_bytes / 16, uint32_t(it));
                        KAIROS_CUDA_TRY(cudaGetLastError());
                    }
                    const int r = it - warmup;
                    if (r >= 0) KAIROS_CUDA_TRY(cudaEventRecord(events.ev[2 * r], stream));
                    if (int rc = mixed_step_impl(ctx, B, q_dec, dpt, stride, lens.data(), C, prefix_len, q_chunk, cpt,
                                                 int32_t(std::max<int64_t>(cp, 1)), o_dec, o_chunk, nullptr, nullptr, stream))
                        return rc;
                    if (r >= 0) KAIROS_CUDA_TRY(cudaEventRecord(events.ev[2 * r + 1], stream));
                }
                if (cudaStreamSynchronize(stream) != cudaSuccess) {
                    const cudaError_t ce = cudaGetLastError();
                    return fail(KAIROS_ERR_CUDA, std::string("latency table: step failed on the device: ") + cudaGetErrorString(ce));
                }
                times.clear();
                for (int r = 0; r < reps; ++r) {
                    float ms = 0.f;
                    KAIROS_CUDA_TRY(cudaEventElapsedTime(&ms, events.ev[2 * r], events.ev[2 * r + 1]));
                    times.push_back(double(ms) * 1e3);
                }
                std::sort(times.begin(), times.end());
                const size_t n = times.size();
                out_median_us[o] = n % 2 ? times[n / 2] : 0.5 * (times[n / 2 - 1] + times[n / 2]);
                if (out_min_us) out_min_us[o] = times[0];
            }
    return KAIROS_OK;
}
