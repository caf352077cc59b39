// Internal declarations shared by the translation units of libkairos.so (never installed).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "kairos.h"

namespace kairos {

constexpr int kHeads = 16;
constexpr int kLatent = 512;
constexpr int kRope = 64;
constexpr int kDim = 576;             // latent | rope
constexpr int kPage = 64;
constexpr int kTokenBytes = kDim * 2; // 1152

// ---- error plumbing -------------------------------------------------------------------------------
void set_error(const std::string& msg);
int fail(int code, const std::string& msg);
#define KAIROS_CUDA_TRY(expr)                                                                            \
    do {                                                                                                 \
        cudaError_t _e = (expr);                                                                         \
        if (_e != cudaSuccess)                                                                           \
            return ::kairos::fail(KAIROS_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(_e));  \
    } while (0)

// ---- work items: what one CTA pass of the attention kernel processes ---------------------------------
// kind 0 = decode split (1 query token x 16 heads over pages [page_begin, page_end) of its sequence),
// kind 1 = chunk tile (kChunkTokens query tokens x 16 heads over pages [0, page_end), causal).
struct WorkItem {
    int32_t kind;        // 0 decode split, 1 chunk tile
    int32_t q_index;     // decode: request index; chunk: first query token of the tile
    int32_t page_begin;  // first logical page of the KV range
    int32_t page_end;    // one past the last logical page
    int32_t n_keys;      // decode: L_i; chunk: P + q_index + 1 (keys visible to the tile's first token)
    int32_t n_q;         // query tokens in this item (decode 1; chunk <= kChunkTokens, ragged tail)
    int32_t partial_slot; // >= 0: write unnormalised partial (o, m, l) to this workspace slot; -1: final output
    int32_t cost;        // planner's cost estimate (pages-equivalents), used for ordering only
};
static_assert(sizeof(WorkItem) == 32, "WorkItem is copied to the device as raw bytes");

// One entry per decode request that was split: the combine pass merges n_splits partial slots.
struct CombineItem {
    int32_t q_index;      // output token: decode request index, or chunk token index
    int32_t first_slot;   // first partial slot of this token
    int32_t n_splits;
    int32_t kind_stride;  // bits 0..7: 0 decode / 1 chunk output; bits 8..: slot stride between splits
};

struct Plan {
    std::vector<WorkItem> items;       // execution order (longest first)
    std::vector<CombineItem> combines;
    std::vector<WorkItem> pair_items;  // chunk tiles of 8 tokens for the 2-CTA pair kernel (empty: chunk runs as gen-1 tiles)
    int32_t n_pairs = 0;               // clusters the pair kernel is launched with (one per SM pair, at most one per tile)
    int32_t dec_ctas = 0;              // with n_pairs > 0: CTAs of the decode grid launched BEFORE the clusters (even); 0 = one per SM, behind them
    int32_t n_decode_items = 0;
    int32_t n_chunk_items = 0;
    int32_t n_partial_slots = 0;
};

// Host planner (a0): pure integer code, no CUDA.  `target_ctas` = resident CTAs the launch will have.
// chunk_tile_tokens = query tokens per chunk tile.  pair_mode: 0 = chunk as gen-1 tiles in the same queue, -1 = let the
// planner decide whether (and on how many SM pairs) the chunk runs on the pair kernel, n > 0 = force n pairs.  See plan.cpp.
void build_plan(const int32_t* dec_ctx_lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len,
                int32_t target_ctas, int32_t chunk_tile_tokens, Plan* plan, int32_t pair_mode = 0,
                int32_t pair_tile_tokens = 8);

constexpr size_t kPartialSlotBytes = size_t(kHeads) * kLatent * 4 + size_t(kHeads) * 2 * 4;  // o[16][512] f32 + (m,l)[16]

// ---- context ---------------------------------------------------------------------------------------
struct HostStage {  // device staging for kairos_mixed_step_host
    void* dev = nullptr;
    size_t bytes = 0;
    cudaStream_t in = nullptr, out = nullptr;  // a sliced step's H2D / D2H copies run here, beside the attention on the caller's stream
    std::vector<cudaEvent_t> events;           // [2i] slice i's queries are up, [2i + 1] slice i's step is done
};

struct StepArgs {
    int32_t n_dec;
    const void* q_dec;
    const int32_t* dec_page_tables;
    int32_t dec_table_stride;
    int32_t chunk_len, prefix_len;
    const void* q_chunk;
    const int32_t* chunk_page_table;
    void* out_dec;
    void* out_chunk;
    float* lse_dec;
    float* lse_chunk;
    int32_t fp8 = 0;  // 1: kairos_fp8_decode (decodes only, over the attached fp8 pool)
};

// Device-resident copy of one plan's work lists (items | combines | pair items) with its pinned source.
struct PlanBuffer {
    void* host = nullptr;              // pinned
    void* dev = nullptr;
    size_t cap = 0;
    cudaEvent_t uploaded = nullptr;    // recorded behind the H2D copy out of `host`
    cudaEvent_t last_use = nullptr;    // recorded on the caller's stream behind the kernels that read `dev`
    bool upload_pending = false;       // the H2D may still be in flight: the caller's stream waits on `uploaded`
    bool ever_used = false;
    cudaGraphExec_t exec = nullptr;    // the step's kernels captured for `gargs` (replayed by cudaGraphLaunch)
    StepArgs gargs{};
    int same_args_uses = 0;            // consecutive uses with the pointer set of `gargs`
};

// One cached plan (a0): reused by every later step with the same (lengths, C, P) without planning, copying or encoding
// anything (exact hit), or -- when only lengths inside the last pages moved, so that every request keeps its page count --
// patched in place and re-uploaded to the other buffer (structural hit).
struct PlanEntry {
    bool valid = false;
    uint64_t stamp = 0;                // LRU clock
    int32_t n_dec = 0, chunk_len = 0, prefix_len = 0, target_ctas = 0, pair_mode = 0, fp8 = 0;
    std::vector<int32_t> lens;
    Plan plan;
    size_t items_bytes = 0, comb_off = 0, comb_bytes = 0, pair_off = 0, pair_bytes = 0, total_bytes = 0;
    PlanBuffer buf[2];
    int cur = 0;
};

// kairos_fp8_attach: the fp8 pool and its tensor maps
struct Fp8State {
    bool attached = false;
    void* pool8 = nullptr;
    int32_t num_pages = 0;
    CUtensorMap lat_map, rope_map;
};

// kairos_run_schedule: the plans of every step of the last schedule, their device copies and the captured graph
struct ScheduleCache {
    std::vector<uint8_t> key;          // every argument, length and chunk size of the schedule the graph was captured for
    std::vector<PlanEntry> steps;
    std::vector<size_t> plan_off;
    size_t pos_off = 0;
    void* host = nullptr;              // pinned arena: work lists of every step | append positions of the decodes
    void* dev = nullptr;
    size_t cap = 0;
    cudaGraphExec_t exec = nullptr;
    int kernels = 0;
};

// kairos_tune_step: the launch order measured fastest for a step shape (page counts per decode, C, P)
struct TunedShape {
    uint64_t key = 0;      // hash of (n_dec, page count of every decode, chunk_len, prefix pages)
    int32_t pair_mode = -1;
};

struct QMapCache {  // a tensor map stays valid while (pointer, rows) do not change
    const void* ptr = nullptr;
    uint64_t rows = 0;
    CUtensorMap map;
};

}  // namespace kairos

struct kairos_ctx {
    kairos_config cfg;
    int sm_count = 0;
    CUtensorMap pool_map;         // TMA descriptor of the pool (placeholder q map when a side of the step is empty)
    CUtensorMap pool_map2, pool_map1;  // boxes of 2 latent chunks / 1 chunk of a page: the slot ring of kairos_mixed_kernel
    CUtensorMap pool_map_c;       // a group of 64-dim chunks of a page: K ring of the pair kernel's S-CTA
    CUtensorMap pool_map_v;       // latent part of a page (box of 8 chunks): V operand of the pair kernel
    kairos::QMapCache proj_a[2], proj_b[2];    // operand maps of kairos_absorb_q [0] and kairos_project_out [1]
    kairos::QMapCache qs_map;                  // decode q of kairos_decode_static (its own cache: the other paths' maps stay as they are)
    kairos::QMapCache qd_map, qc_map, qp_map;  // decode q (box 16 rows), chunk q for gen-1 tiles (64 rows), for the pair kernel (128 rows)
    cudaStream_t copy_stream = nullptr;   // plan H2D copies run here, beside whatever precedes the step on the caller's stream
    cudaStream_t capture_stream = nullptr;  // the step's launches are captured here when a plan is replayed as a CUDA graph
    // kairos_debug_set knobs (tests and sweeps only)
    int force_pairs = -1;         // -1 auto, 0 never use the pair kernel, n > 0 decode grid first beside n clusters, -(n + 1) n clusters first
    int force_dec_only = -1;      // 0 = never use the decode-only instantiation
    int use_copy_stream = 1, use_graph = 1, use_plan_cache = 1;
    int host_slice_tokens = 0;    // kairos_mixed_step_host: 0 = its own rule, n > 0 = slices of n chunk tokens
    std::vector<kairos::TunedShape> tuned;   // filled by kairos_tune_step; consulted when force_pairs == -1
    static constexpr int kPlanEntries = 12;  // a sliced host step alone uses up to 8 (7 slices + the decodes' step)
    kairos::PlanEntry plans[kPlanEntries];
    uint64_t plan_clock = 0;
    kairos::HostStage host_stage;
    kairos::ScheduleCache schedule;
    int64_t last_info[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    bool profile = false;         // bracket the attention kernels with events (kairos_profile_enable)
    std::vector<cudaEvent_t> prof_events;  // pairs: [2i] start, [2i+1] stop
    size_t prof_used = 0;         // events in use since the last kairos_profile_read
    // latency-table scratch (allocated once, grown on demand; freed by kairos_destroy)
    void* table_buf = nullptr;
    size_t table_bytes = 0;
    void* flush_buf = nullptr;
    kairos::Fp8State fp8;
};

namespace kairos {

// Shared by kairos_mixed_step, the latency table and the schedule runner: validate, plan (or reuse), stage, launch.
int mixed_step_impl(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                    const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len, const void* q_chunk,
                    const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec, void* out_chunk, float* lse_dec,
                    float* lse_chunk, cudaStream_t stream, int32_t fp8 = 0);

// ---- kernel launchers (each returns a kairos_status) -----------------------------------------------
int launch_append(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens, const int32_t* page_table,
                  int32_t start_pos, cudaStream_t stream);
int launch_append_decode(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n, const int32_t* page_tables,
                         int32_t table_stride, const int32_t* positions, cudaStream_t stream);
int launch_gather(kairos_ctx* ctx, const int32_t* page_table, int32_t n_tokens, void* out, cudaStream_t stream);

// persistent tcgen05/TMA kernel over the plan's work items + LSE combine (attn_umma.cu)
int umma_chunk_tile_tokens();
int umma_resident_ctas(const kairos_ctx* ctx);
int encode_q_map(QMapCache* cache, const void* ptr, uint64_t rows, uint32_t box_rows);  // no-op when (ptr, rows) are unchanged
// bf16 matrix [rows][inner] with `row_stride_bytes` between rows, boxes of box_inner x box_rows, SWIZZLE_128B (cached like encode_q_map)
int encode_2d_map(QMapCache* cache, const void* ptr, uint64_t inner, uint64_t rows, uint64_t row_stride_bytes, uint32_t box_inner,
                  uint32_t box_rows);
int launch_attn_umma(kairos_ctx* ctx, const Plan& plan, const StepArgs& a, const WorkItem* dev_items, int32_t n_items,
                     cudaStream_t stream, int max_ctas, bool as_clusters, bool pdl);
int launch_decode_static(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                         const int32_t* dec_ctx_lens, void* out_dec, float* lse_dec, cudaStream_t stream);
int launch_combine(kairos_ctx* ctx, const StepArgs& a, const CombineItem* dev_combines, int32_t n_combines, cudaStream_t stream);
int umma_init(kairos_ctx* ctx);  // builds tensor maps, sets kernel attributes

// projections either side of the attention (proj.cu)
int launch_absorb_q(kairos_ctx* ctx, const void* q_nope, const void* q_rope, const void* w_uk_t, int32_t n, void* q_out, cudaStream_t stream);
int launch_project_out(kairos_ctx* ctx, const void* o_lat, const void* w_uv_t, int32_t n, void* v_out, cudaStream_t stream);

// fp8 latent cache (fp8.cu)
// tensor map of rank 2 or 3 over bytes (u8) or bf16 elements, SWIZZLE_128B; strides in bytes for dimensions 1..rank-1
int encode_tiled_map(CUtensorMap* out, bool u8, int rank, const void* ptr, const uint64_t* dims, const uint64_t* strides, const uint32_t* box);
int fp8_attach(kairos_ctx* ctx, void* pool8, int32_t num_pages);
int launch_fp8_append(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens, const int32_t* page_table,
                      int32_t start_pos, cudaStream_t stream);
int launch_fp8_append_decode(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n, const int32_t* page_tables,
                             int32_t table_stride, const int32_t* positions, cudaStream_t stream);
int launch_fp8_decode(kairos_ctx* ctx, const StepArgs& a, const WorkItem* dev_items, int32_t n_items, cudaStream_t stream);

// chunk tiles on 2-CTA clusters (attn_pair.cu)
int pair_tile_tokens();
int pair_init(kairos_ctx* ctx);
int launch_attn_pair(kairos_ctx* ctx, const StepArgs& a, const WorkItem* dev_items, int32_t n_items, int32_t n_pairs,
                     cudaStream_t stream, bool pdl);

}  // namespace kairos
