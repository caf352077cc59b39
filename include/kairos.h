/*
 * kairos.h -- C ABI of libkairos.so: the decode-node mixed attention step that KAIROS creates when it
 * deflects a prefill (arxiv 2607.02043), B200 / sm_100a only.
 *
 * What the step is (section 3.2 methodology; section 5.4): one batch
 * holding B in-flight decodes (one query token each over its own K cached tokens) plus the tokens of one
 * prefill chunk of a deflected request (causal over its already-cached prefix plus the chunk).  "The KV
 * cache is built directly on the decode node", i.e. the chunk's keys are appended to
 * the node's paged cache and read from it.  Per-step latency as a function of (decode batch, cached
 * tokens, chunk size) is the input of the TBT-safety check and chunk-schedule sweep (PAPER.md:253-269,
 * Eq. 4-6; profiled once per model/hardware).
 *
 * The paper leaves the attention kernel unmodified and unspecified; shapes and arithmetic
 * are fixed by BASELINE.json north_star / configs[0] and restated in SURVEY.md 8(c):
 *   absorbed MLA, 16 heads; each cached token = 512-d latent c_t + 64-d RoPE key kR_t shared by all heads;
 *   query row (token j, head h) = [qC (512) | qR (64)];  s_t = scale * (qC.c_t + qR.kR_t);
 *   p = softmax over the visible positions;  o = sum_t p_t c_t (512-d);  lse = ln sum_t exp(s_t).
 *   decode i sees positions 0..L_i-1 (its newest token already appended); chunk row j sees 0..P+j.
 *   bf16 inputs, fp32 accumulation, bf16 outputs, fp32 lse.
 *
 * Memory layout (part of the contract; the append check compares raw pool bytes):
 *   pool       device bf16 [num_pages][64][576]; token slot = pool + ((page*64 + slot)*576)*2 bytes,
 *              512 latent values then 64 RoPE-key values.  Must be 128-byte aligned.
 *   page table int32, entry b = physical page of tokens 64b .. 64b+63 of that sequence.
 *   q          bf16 [n][16][576], row = [latent part 512 | rope part 64], 16-byte aligned.
 *   out        bf16 [n][16][512], 16-byte aligned; lse fp32 [n][16].
 * Precondition on the pool: slots at positions >= the attended length never influence a result, whatever FINITE
 * or NON-FINITE bit pattern they hold (the kernels zero the invisible rows of a boundary page in shared memory
 * before the PV product, so a NaN/Inf left by an allocator cannot reach an output through 0 * NaN).  Visible
 * slots must hold finite values.
 *
 * Ownership: the caller owns every buffer it passes (pool, workspace, q, out, page tables) and the CUDA
 * stream; the context owns only its descriptors, a small pinned staging area and its plan buffers.  No
 * pointer is retained past the call that received it, except `pool` / `workspace` given at create time.
 *
 * Asynchrony: kairos_append_latent and kairos_mixed_step enqueue on `cuda_stream` (a cudaStream_t cast to
 * void*; NULL = legacy default stream) and return without synchronising.  The stream must not be in capture
 * mode (the library replays its own CUDA graphs, see below; kairos_run_schedule builds one for a whole chunk
 * schedule).  Host arrays (dec_ctx_lens) are read before the call returns.  Calls on one context must be issued from one thread at a time and on
 * one stream at a time (the plan buffers are reused per call, ordered by that stream).  Stream order is
 * what the caller sees: a later operation on `cuda_stream` observes every output of an earlier call.  Inside
 * that order the library overlaps its own work: the step's work list is copied on a stream of the context,
 * and kernels are launched with programmatic stream serialisation (a grid may become resident while its
 * predecessor drains, and waits for it on the device before touching anything the predecessor may still use).
 *
 * Plan reuse: the context keeps the last few host plans (a0) with their device copies.  A step whose
 * (n_dec, dec_ctx_lens, chunk_len, prefix_len) match a kept plan skips the planner and the host->device copy; when
 * it also passes the same buffers as the previous use of that plan, its kernels are replayed as one CUDA graph
 * (programmatic launch edges kept).  A step that only moved lengths inside the requests' last pages re-uses the
 * plan's structure (lengths patched, one small copy).  Results never depend on which path was taken.
 *
 * Errors: every call returns 0 (KAIROS_OK) or a negative kairos_status.  Argument errors (NULL pointers, sizes,
 * lengths, misaligned q / out / lse pointers) are detected on the host before anything is enqueued.  Page ids are trusted (not range-checked on the device).
 * kairos_last_error gives a human-readable message for the last failure on this thread.
 * There is no CPU fallback anywhere: without a CUDA device every compute entry returns KAIROS_ERR_CUDA.
 */
#ifndef KAIROS_H_
#define KAIROS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    KAIROS_OK = 0,
    KAIROS_ERR_INVALID_ARG = -1,
    KAIROS_ERR_UNSUPPORTED = -2, /* dims other than 16 / 512 / 64 / page 64, or not an sm_100 device */
    KAIROS_ERR_WORKSPACE = -3,   /* workspace too small for this call: see kairos_workspace_bytes */
    KAIROS_ERR_CUDA = -4         /* a CUDA runtime / driver call failed (message has the CUDA string) */
} kairos_status;

typedef struct kairos_ctx kairos_ctx; /* opaque, owned by the library */

typedef struct {
    int32_t num_heads;     /* must be 16  */
    int32_t latent_dim;    /* must be 512 */
    int32_t rope_dim;      /* must be 64  */
    int32_t page_size;     /* must be 64  */
    float softmax_scale;   /* 1/sqrt(192) for DeepSeek-V2-Lite; any finite > 0 accepted */
    void* pool;            /* DEVICE bf16 [num_pages][64][576], caller-owned, 128-B aligned */
    int32_t num_pages;     /* >= 1 */
    void* workspace;       /* DEVICE scratch, caller-owned, 256-B aligned; split-KV partials live here */
    size_t workspace_bytes;
    int32_t device;        /* CUDA device ordinal the buffers live on */
} kairos_config;

/* Bytes of device workspace that are always enough for a step with <= max_decodes decodes and a chunk of
 * <= max_chunk tokens (host-only arithmetic, no CUDA call). */
size_t kairos_workspace_bytes(int32_t max_decodes, int32_t max_chunk);

/* Validates the config, builds the TMA descriptor of the pool, allocates plan/staging buffers.
 * *out is set only on success.  HOST pointers: cfg, out. */
int kairos_create(const kairos_config* cfg, kairos_ctx** out);
int kairos_destroy(kairos_ctx* ctx); /* NULL is a no-op */

/*
 * a1 -- paged latent-cache append ("the cache is built directly on the decode node").
 * Copies latent[j][0:512] | k_rope[j][0:64] to the slot of position start_pos + j, j < n_tokens, of the
 * sequence whose page table is `page_table`.  Bit-exact byte copy, 16-byte vector stores.
 *   latent      DEVICE bf16 [n_tokens][512], 16-B aligned     k_rope  DEVICE bf16 [n_tokens][64], 16-B aligned
 *   page_table  DEVICE int32 [table_len]
 * Errors: INVALID_ARG if n_tokens < 0, start_pos < 0, a pointer is NULL with n_tokens > 0, or
 * start_pos + n_tokens > table_len*64.  n_tokens == 0 is a successful no-op.
 */
int kairos_append_latent(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens,
                         const int32_t* page_table, int32_t table_len, int32_t start_pos, void* cuda_stream);

/*
 * Batched single-token append for the decodes of a step: request i writes one token at position
 * positions[i] through row i of page_tables.
 *   latent DEVICE bf16 [n][512]; k_rope DEVICE bf16 [n][64]; page_tables DEVICE int32 [n][table_stride];
 *   positions DEVICE int32 [n], each in [0, table_stride*64).  (positions are trusted: device-side only.)
 */
int kairos_append_decode_tokens(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n,
                                const int32_t* page_tables, int32_t table_stride, const int32_t* positions,
                                void* cuda_stream);

/* Test/inspection export: walks `page_table` and copies positions 0..n_tokens-1 out, bit-exact.
 *   out DEVICE bf16 [n_tokens][576].  Errors as for append (n_tokens > table_len*64 -> INVALID_ARG). */
int kairos_gather_latent(kairos_ctx* ctx, const int32_t* page_table, int32_t table_len, int32_t n_tokens,
                         void* out, void* cuda_stream);

/*
 * The mixed step: n_dec decode queries plus one causal prefill chunk, one launch sequence.
 *   q_dec            DEVICE bf16 [n_dec][16][576]
 *   dec_page_tables  DEVICE int32 [n_dec][dec_table_stride]
 *   dec_ctx_lens     HOST   int32 [n_dec], each >= 1 and <= dec_table_stride*64 (attended length L_i)
 *   chunk_len        C >= 0 prefill tokens in this step; prefix_len P >= 0 tokens of the same request
 *                    already cached; the chunk's own C tokens must have been appended at positions
 *                    P..P+C-1 earlier on the same stream
 *   q_chunk          DEVICE bf16 [C][16][576]
 *   chunk_page_table DEVICE int32 [chunk_table_len], chunk_table_len*64 >= P + C
 *   out_dec          DEVICE bf16 [n_dec][16][512]     out_chunk DEVICE bf16 [C][16][512]
 *   lse_dec          DEVICE fp32 [n_dec][16] or NULL  lse_chunk DEVICE fp32 [C][16] or NULL
 * n_dec == 0 and chunk_len == 0 together are a successful no-op.  Exactly one chunk per step (the
 * dispatcher sends a decode node one deflected request at a time).
 * Errors: INVALID_ARG (negative sizes, NULL where data is needed, ctx_len < 1 or beyond its table,
 * chunk table too short), WORKSPACE (workspace smaller than this step's split-KV partials need).
 */
int kairos_mixed_step(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                      int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len,
                      const void* q_chunk, const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec,
                      void* out_chunk, float* lse_dec, float* lse_chunk, void* cuda_stream);

/*
 * The same step driven from HOST buffers (end-to-end leg): copies q_dec, q_chunk, the page tables and the
 * chunk's new latent / k_rope host->device (pinned or pageable host memory), appends the chunk at
 * prefix_len, runs the mixed step, copies out_dec / out_chunk (and lse if non-NULL) device->host, and
 * synchronises the stream before returning.  All pointers are HOST pointers with the shapes of
 * kairos_mixed_step / kairos_append_latent; device staging comes from the context (grown on demand).
 * h2d_bytes / d2h_bytes (HOST, may be NULL) receive the bytes copied each way.
 * A chunk of at least two rounds of the cluster grid (2 * (SMs / 2) * 8 tokens, 1184 on a B200) is cut into at most 7
 * slices of whole rounds that run as successive mixed steps over a growing prefix (the same tiles over the same keys:
 * chunk invariance; the whole chunk is appended first, the decodes run ahead as a step of their own), with the next
 * slice's queries copied up and the previous slice's outputs copied down on two streams of the context beside the
 * attention on `cuda_stream`: the PCIe copies (34.8 KB per chunk token) overlap the step instead of bracketing it.
 * Host buffers should be pinned for that overlap (pageable memory works, without it).  Nothing is left in flight on return.
 */
int kairos_mixed_step_host(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                           int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len,
                           int32_t prefix_len, const void* q_chunk, const void* chunk_latent, const void* chunk_k_rope,
                           const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec, void* out_chunk,
                           float* lse_dec, float* lse_chunk, uint64_t* h2d_bytes, uint64_t* d2h_bytes,
                           void* cuda_stream);

/*
 * a11 -- per-step latency table over a (decode batch B, per-decode context K, chunk size C) grid: the
 * deployment-time profiling of PAPER.md:302-304 for this one layer's attention, the input of Eq. 4-6
 * (PAPER.md:253-269).  For every (B, K, C): synthetic page tables over the context's pool (B*ceil(K/64) +
 * ceil((prefix_len+C)/64) distinct pages, strided through the pool), `warmup` untimed steps, then `reps`
 * timed steps (one CUDA event pair per rep around kairos_mixed_step on `cuda_stream`; when flush_l2 != 0 a buffer
 * larger than L2 is rewritten before every step, outside the timed interval).  The reps of a point are enqueued back
 * to back and read after one synchronisation, so with warmup >= 2 an interval is the DEVICE time of the step (the
 * cached plan's graph is already queued when the start event fires); warmup < 2 puts the planner and the plan copy
 * of the first use inside the first interval.  The chunk's tokens are not appended (timing only: the pool's bytes
 * are read as they are).  Scratch buffers belong to the context and are allocated on first use.  Synchronising call.
 *   Bs, Ks, Cs         HOST int32 arrays (B >= 0, K >= 1, C >= 0; B == 0 and C == 0 together give 0 us)
 *   out_median_us      HOST double [nB*nK*nC], index (iB*nK + iK)*nC + iC
 *   out_min_us         HOST double [nB*nK*nC] or NULL
 * Units: K is PER-DECODE context (the paper's K_n is total occupancy = B*K); C is prefill tokens only (the
 * paper's chi counts B + C); entries are one layer's attention in microseconds (SURVEY.md 8(b) units note).
 * Errors: INVALID_ARG; WORKSPACE if the pool has too few pages or the workspace is too small for a point.
 */
int kairos_step_latency_table(kairos_ctx* ctx, const int32_t* Bs, int32_t nB, const int32_t* Ks, int32_t nK,
                              const int32_t* Cs, int32_t nC, int32_t prefix_len, int32_t warmup, int32_t reps,
                              int32_t flush_l2, double* out_median_us, double* out_min_us, void* cuda_stream);

/*
 * a0 -- the host planner alone (no GPU, no context): the work list kairos_mixed_step would build for these
 * lengths on a device with `n_ctas` resident CTAs.  Pure integer host code; used by the CPU tests to check that
 * every (request, page) and every chunk token is covered exactly once and that the partial slots stay inside the
 * kairos_workspace_bytes bound.
 *   dec_ctx_lens   HOST int32 [n_dec] (each >= 1)
 *   pair_mode      0 = the chunk runs as 4-token tiles in the same queue as the decode splits; -1 = the planner
 *                  decides whether the chunk runs as 8-token tiles on 2-CTA clusters that share the SMs in time with
 *                  the decode grid, and in which order the two grids are launched, as kairos_mixed_step does
 *                  (DESIGN.md 6.2); n > 0 = the decode grid first, beside n resident clusters (n >= every SM pair:
 *                  the clusters first); -(n + 1) = n clusters first, the decode grid on every SM behind them
 *   items_out      HOST int32 [max_items][8]: kind (0 decode split / 1 chunk tile in the queue / 2 chunk tile of the
 *                  cluster kernel), q_index (request index or first chunk token), page_begin, page_end, n_keys, n_q,
 *                  partial_slot (-1 = final output), cost; queue order, then the cluster kernel's items.  May be NULL.
 *   n_items_out    HOST, number of items of the plan (even if > max_items; only max_items are written)
 *   n_partial_slots_out, n_pairs_out  HOST or NULL (clusters the cluster kernel would be launched with; 0 = unused)
 * Errors: INVALID_ARG.
 */
int kairos_plan_dump(const int32_t* dec_ctx_lens, int32_t n_dec, int32_t chunk_len, int32_t prefix_len, int32_t n_ctas,
                     int32_t pair_mode, int32_t* items_out, int32_t max_items, int32_t* n_items_out,
                     int32_t* n_partial_slots_out, int32_t* n_pairs_out);

/* Introspection of the last kairos_mixed_step plan on this context -- after kairos_run_schedule: the plan of the schedule's
 * LAST step, with [4] = every kernel of the whole schedule, appends included -- (host-only; for tests, bench):
 * info[0] = work items, [1] = decode splits, [2] = chunk tiles, [3] = CTAs launched, [4] = kernels launched
 * by that call, [5] = workspace bytes used, [6] = 2-CTA clusters the chunk ran on (0 = the chunk ran as tiles of the
 * decode grid's queue), [7] = plan cache (0 planned, 1 structure re-used with patched lengths, 2 exact hit),
 * [8] = 1 if the kernels were replayed as a CUDA graph, [9] = CTAs of the decode grid when it is launched before the
 * clusters (0 otherwise).  n = number of int64 slots available in info (at most 10 are written). */
int kairos_last_plan_info(const kairos_ctx* ctx, int64_t* info, int32_t n);

/*
 * Kernel-level timing for the roofline leg of bench.py.  While enabled, kairos_mixed_step brackets the launch of
 * its main (persistent attention) kernel with a pair of CUDA events on the caller's stream.  kairos_profile_read
 * synchronises the recorded events, returns the summed main-kernel device time in microseconds and the number of
 * launches since the last read (HOST pointers, either may be NULL), and clears the record.
 */
int kairos_profile_enable(kairos_ctx* ctx, int32_t on);
int kairos_profile_read(kairos_ctx* ctx, double* main_kernel_us_total, int64_t* launches);

/* ------------------------------------------------------------------------------------------------------------
 * the consumer of the latency table: KAIROS' step-latency model, TBT-safe chunk schedule and
 * deflection decision (section 4.2-4.4, Eq. 1-7; Algorithm 1).  Pure HOST code: no CUDA
 * call, no context; every pointer below is a HOST pointer; all latencies are in the unit of the samples the model was
 * fitted on (microseconds when they come from kairos_step_latency_table).
 *
 * Eq. 4: T_step = T0 + dT_pf, both "simple linear regressors" fitted once per model/hardware
 * (PAPER.md:302-313).  The paper lumps all cached tokens into K_n; one attention layer treats a decode's cached token
 * (read once per step) and a cached token of the deflected request (met by every query token of the chunk) differently,
 * so the model keeps them apart (reading G20):
 *     T0(B, Kd)       = a[0] + a[1]*B + a[2]*Kd                              Kd = tokens cached by the B in-flight decodes
 *     dT_pf(C, P, Kd) = b[0] + b[1]*C + b[2]*C*(P + (C+1)/2) + b[3]*Kd       C > 0 prefill tokens over a P-token prefix
 *     dT_pf = 0 for C = 0.
 * Prefill-node step latency: T_pf_step(tokens, cached) = p[0] + p[1]*tokens + p[2]*cached + p[3]*tokens*cached.
 */
typedef struct {
    double a[3];
    double b[4];
} kairos_step_model;

typedef struct {
    double p[4];
} kairos_prefill_model;

/*
 * Closed-form weighted least squares for the two regressors of Eq. 4, as PAPER.md:312 describes: T0 from the samples
 * with C == 0, then dT_pf from the residual T - T0 of the samples with C > 0.  Rows are weighted by 1/T so that the
 * fit minimises relative error, the criterion the paper states (MAPE < 10 %; reading G21).
 *   B, Kd, C, P   int64 [n]    sample points (Kd = B * K for a table entry with per-decode context K)
 *   T             double [n]   measured step latency, each > 0
 *   model         out
 *   mape_out      out or NULL: mean |pred - T| / T over the n samples
 * Errors: INVALID_ARG (NULL, n < 1, T <= 0, fewer than 3 decode-only or 4 mixed samples, or a singular system, e.g.
 * every sample with the same B).
 */
int kairos_fit_latency_model(const int64_t* B, const int64_t* Kd, const int64_t* C, const int64_t* P, const double* T,
                             int32_t n, kairos_step_model* model, double* mape_out);

/* Eq. 4 evaluated: predicted latency of a step with B decodes caching Kd tokens and C prefill tokens over a P-token prefix. */
double kairos_predict_step(const kairos_step_model* model, int64_t B, int64_t Kd, int64_t C, int64_t P);

typedef struct {
    int32_t prompt_len;          /* l_r >= 1 */
    const int32_t* queue_lens;   /* prompt lengths queued ahead of r on its prefill node (FIFO), [n_queue] */
    int32_t n_queue;
    int32_t chi_p;               /* prefill-node chunk size >= 1 */
    const int32_t* node_B;       /* decode-node states: B_n in-flight decodes ...            [n_nodes] */
    const int64_t* node_K;       /* ... caching K_n tokens in total                          [n_nodes] */
    int32_t n_nodes;
    const int32_t* candidates;   /* chunk-size candidates chi_1 > ... > chi_C > 0: TOTAL tokens of a step (the paper's
                                    chi), of which chi - B_n are prefill tokens     [n_candidates] */
    int32_t n_candidates;
    double tbt_slo;              /* tau */
    double beta;                 /* safety factor of Eq. 5, > 0 */
    double alpha;                /* deflection margin of Eq. 7, >= 1 */
    double ttft_slo;
} kairos_decide_input;

typedef struct {
    int32_t decision;            /* 0 = KEEP on the prefill node, 1 = DEFLECT */
    int32_t node;                /* n* (index into node_B / node_K), -1 when kept */
    int32_t n_steps;             /* |X*|, 0 when kept */
    double ttft_pf;              /* Eq. 1 */
    double ttft_dec;             /* Eq. 6 of the fastest feasible node (+inf if none is feasible) */
} kairos_decide_output;

/*
 * Algorithm 1: (1) prefill-node TTFT estimate, Eq. 1-3; (2) for every decode node the greedy TBT-safe
 * schedule X = [chi(1) .. chi(m)] -- at each step the largest candidate with T_step <= beta * tau (Eq. 5) -- and its
 * TTFT estimate (Eq. 6); (3) the fastest feasible node; (4) DEFLECT iff Eq. 7 holds.  Readings of the garbled spots
 * (G19): Eq. 3 sums i = 0 .. ceil(l_r/chi_p) - 1; a step serves chi - B_n prefill tokens, candidates <= B_n
 * are skipped; the feasible set starts empty; the threshold is beta * tau.  State projected for step i of a schedule on
 * node n: Kd = K_n + (i-1)*B_n, P = prefill tokens served so far, C = chi(i) - B_n.  Ties between nodes go to the lowest index.
 *   schedule_out   int32 [max_schedule] or NULL: X* (the chi values, in order).  kairos_run_schedule takes the prefill
 *                  tokens per step, chi(i) - B_n (the last one trimmed to what is left of the prompt).
 * Never returns DEFLECT for a schedule the model predicts unsafe.  Cost: O(n_nodes * ceil(l_r /
 * (chi_min - B)) * n_candidates) evaluations of Eq. 4.
 * Errors: INVALID_ARG (NULL, sizes < 1, candidates not strictly decreasing, beta <= 0, alpha < 1), WORKSPACE if X* is
 * longer than max_schedule (out->n_steps holds the length needed).
 */
int kairos_decide(const kairos_step_model* model, const kairos_prefill_model* prefill, const kairos_decide_input* in,
                  int32_t* schedule_out, int32_t max_schedule, kairos_decide_output* out);

/*
 * SURVEY.md 8(f) row 4 (second half) -- the paper's policy simulator ("we wrap the three predictors in an
 * event-based simulator with support for PD disaggregation"; section 3.4, Table 4): the latency models
 * above inside an event loop over n_prefill FIFO prefill nodes and n_decode decode nodes.  Host only.  The paper prints no
 * pseudo-code for it; the rules (reading G22) are:
 *   - A request that is not deflected goes to the prefill node with the fewest outstanding prompt tokens (ties: lowest
 *     index), occupies it for T_pf (Eq. 3) in FIFO order, and is ready on a decode node transfer_per_token * l_r later
 *     (KV transfer = bytes over bandwidth); its TTFT is that instant minus its arrival.  It joins the decode
 *     node with the fewest in-flight + pending requests at the time its prefill ends.
 *   - A decode node runs steps back to back while it has work.  A step admits the pending requests that are ready, then
 *     runs B in-flight decodes caching Kd tokens plus -- if a deflected request is in its prefill phase there (at most one
 *     per node) -- C = min(max(chi - B, 1), tokens left) of its prompt over the P already served, and lasts
 *     T_step(B, Kd, C, P) (Eq. 4).  At its end every decode has one more token and leaves when its output is complete; a
 *     deflected request whose prompt is complete has TTFT = step end - arrival and decodes on the same node from then on.
 *   - A step with B > 0 longer than tbt_slo is a TBT violation of the step and of every request decoding in it.
 *   - policy 0 Baseline: never deflect.  1 SQ(param): deflect when more than `param` requests WAIT on every prefill node.
 *     2 SL(param): deflect when l_r < param.  Both to the decode node with the fewest in-flight decodes that hosts no
 *     deflected request (none: prefill path), with the fixed chi = static_chi (128 in the paper).  3 Oracle: kairos_decide on
 *     the simulator's own state (the queue of the prefill node the request would take; (B, Kd) of the eligible decode nodes);
 *     the schedule X* is followed step by step, its last chi repeated if it runs out.
 *   - Events at equal times: decode step ends (node order), prefill completions (node order), arrivals; then idle nodes start.
 *   reqs      HOST [n], sorted by arrival; prompt_len >= 1, output_len >= 0 (tokens decoded after the first)
 *   ttft_out  HOST double [n] or NULL
 * Result: deflections, P95 (nearest rank) and mean TTFT, decode steps and those over tbt_slo, SLO attainment (TTFT <= ttft_slo
 * and no violated step), makespan -- Table 4's columns.  Errors: INVALID_ARG.
 */
typedef struct {
    double arrival;
    int32_t prompt_len;
    int32_t output_len;
} kairos_sim_request;

typedef struct {
    int32_t n_prefill, n_decode;
    int32_t chi_p;               /* prefill-node chunk size */
    int32_t policy;              /* 0 baseline, 1 SQ(theta), 2 SL(l), 3 Oracle */
    int32_t param;               /* theta or l */
    int32_t static_chi;          /* chi of the static policies (total tokens per step) */
    const int32_t* candidates;   /* Oracle: chunk-size candidates, strictly decreasing */
    int32_t n_candidates;
    double tbt_slo, beta, alpha, ttft_slo;
    double transfer_per_token;   /* KV transfer time per prompt token */
} kairos_sim_config;

typedef struct {
    int32_t n_requests, n_deflected;
    double p95_ttft, mean_ttft;
    int64_t decode_steps, tbt_violations;
    double slo_attainment, makespan;
} kairos_sim_result;

int kairos_simulate(const kairos_step_model* model, const kairos_prefill_model* prefill, const kairos_sim_config* cfg,
                    const kairos_sim_request* reqs, int32_t n, double* ttft_out, kairos_sim_result* out);

/*
 * what the decode node does with a deflected request (section 4.3.2;
 * PAPER.md:363-367 section 5.4; Fig. 1's "successive chunks"): the chunk schedule X = [chi(1) ..
 * chi(m)] executed as m successive steps behind one call.  Step i (0-based):
 *   1. if dec_latent != NULL, every in-flight decode j caches its newest token (dec_latent[i][j] | dec_k_rope[i][j]) at
 *      position dec_ctx_lens[j] + i of its sequence and then attends to dec_ctx_lens[j] + i + 1 tokens; with dec_latent ==
 *      NULL the decodes' contexts do not move (each attends to dec_ctx_lens[j] tokens in every step);
 *   2. chunk i of the prompt -- chunk_sizes[i] PREFILL tokens (the paper's chi(i) - B_n) -- is appended at positions
 *      prefix_len + sum_{k<i} chunk_sizes[k] .. of the request's sequence;
 *   3. one mixed step: the n_dec decode queries q_dec[i] plus the chunk's queries, causal over the request's prefix.
 * The whole schedule is planned up front (a0 for every step), its work lists are copied to the device once, and its
 * launches -- appends, attention grids, combines, programmatic edges included -- are captured into ONE CUDA graph that is
 * launched on `cuda_stream`; a call that repeats the previous call's arguments replays the graph.  Results are those of
 * m calls of kairos_append_* / kairos_mixed_step (chunk invariance: the prompt's outputs equal a one-shot
 * causal prefill row for row).
 *   q_dec        DEVICE bf16 [n_steps][n_dec][16][576]      out_dec DEVICE bf16 [n_steps][n_dec][16][512]
 *   dec_page_tables DEVICE int32 [n_dec][dec_table_stride], covering dec_ctx_lens[j] + n_steps tokens when contexts grow
 *   dec_ctx_lens HOST int32 [n_dec]: tokens cached BEFORE the schedule starts (>= 1, or >= 0 when contexts grow)
 *   dec_latent   DEVICE bf16 [n_steps][n_dec][512] or NULL  dec_k_rope DEVICE bf16 [n_steps][n_dec][64] or NULL
 *   chunk_sizes  HOST int32 [n_steps], each >= 1, summing to prompt_len
 *   q_prompt     DEVICE bf16 [prompt_len][16][576]          prompt_latent [prompt_len][512], prompt_k_rope [prompt_len][64]
 *   prompt_page_table DEVICE int32 [prompt_table_len], covering prefix_len + prompt_len tokens
 *   out_prompt   DEVICE bf16 [prompt_len][16][512]          lse_dec [n_steps][n_dec][16] / lse_prompt [prompt_len][16] or NULL
 *   ttft_us      HOST or NULL: measured TTFT_dec of the schedule (the left-hand side of Eq. 6): device time
 *                from the first append to the end of the last step, CUDA events on `cuda_stream`
 *   step_us      HOST double [n_steps] or NULL: device time of every step (this mode launches the steps one by one
 *                with an event pair around each instead of replaying the graph)
 * Asynchronous unless ttft_us or step_us is given (then it synchronises the stream).  A call whose arguments differ from
 * the previous call's synchronises `cuda_stream` once before it overwrites the schedule's device arena.
 * Errors: INVALID_ARG (sizes, NULL, chunk sizes not summing to prompt_len, a page table too short, misaligned buffers),
 * WORKSPACE (a step's split-KV partials exceed the workspace), CUDA.
 */
int kairos_run_schedule(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                        int32_t dec_table_stride, const int32_t* dec_ctx_lens, const void* dec_latent,
                        const void* dec_k_rope, int32_t prompt_len, const int32_t* chunk_sizes, int32_t n_steps,
                        const void* q_prompt, const void* prompt_latent, const void* prompt_k_rope,
                        const int32_t* prompt_page_table, int32_t prompt_table_len, int32_t prefix_len, void* out_dec,
                        void* out_prompt, float* lse_dec, float* lse_prompt, double* step_us, double* ttft_us,
                        void* cuda_stream);

/*
 * the projections either side of the attention (absorbed MLA of DeepSeek-V2-Lite; the
 * math is SURVEY.md 8(c)'s definition): per head h,
 *   kairos_absorb_q     q_out[j][h][0:512]   = sum_k q_nope[j][h][k] * w_uk_t[h][d][k]   (128 -> 512, the key up-projection
 *                       q_out[j][h][512:576] = q_rope[j][h][0:64]                         folded into the query), producing the
 *                       q rows kairos_mixed_step takes;
 *   kairos_project_out  v_out[j][h][e]       = sum_d o_lat[j][h][d] * w_uv_t[h][e][d]    (512 -> 128, the value up-projection)
 *                       applied to kairos_mixed_step's outputs.
 * bf16 operands, fp32 accumulation on tcgen05 (TMEM accumulator), bf16 round-to-nearest-even results.
 *   q_nope  DEVICE bf16 [n][16][128]   q_rope DEVICE bf16 [n][16][64]   w_uk_t DEVICE bf16 [16][512][128]
 *   q_out   DEVICE bf16 [n][16][576]   o_lat  DEVICE bf16 [n][16][512]  w_uv_t DEVICE bf16 [16][128][512]
 *   v_out   DEVICE bf16 [n][16][128]   (all 16-byte aligned; weights are stored [head][output dim][input dim])
 * Asynchronous on `cuda_stream`.  n == 0 is a no-op.  Errors: INVALID_ARG, CUDA.
 */
int kairos_absorb_q(kairos_ctx* ctx, const void* q_nope, const void* q_rope, const void* w_uk_t, int32_t n, void* q_out,
                    void* cuda_stream);
int kairos_project_out(kairos_ctx* ctx, const void* o_lat, const void* w_uv_t, int32_t n, void* v_out, void* cuda_stream);

/*
 * Measured launch order for a step shape.  The host planner (a0) ranks the orders in which the decode grid and the chunk's
 * clusters take the SMs with a cost model; off the workloads it was calibrated on the model can be 10-30 % off the best
 * order (profiles/r02_planner_offpoints.md).  This call runs the step given (same arguments and preconditions as
 * kairos_mixed_step: the chunk already appended) under each candidate order -- the planner's own, every cluster first, a
 * few clusters first, the decode grid first beside n clusters, one queue -- `reps` times each after two warm-ups, timed with
 * CUDA events on `cuda_stream` (it SYNCHRONISES after every run), and pins the fastest for every later kairos_mixed_step /
 * kairos_run_schedule step of this context with the same shape (same number of decodes, same page count per decode, same
 * chunk_len, same number of prefix pages), unless it beats the planner's order by less than 3 %.  Results of every
 * candidate are the same attention outputs (every order is parity-tested); out_dec / out_chunk hold the last run's.
 *   chosen_mode  HOST or NULL: the pinned order in kairos_plan_dump's pair_mode encoding, -1 = the planner's own was kept
 *   chosen_us / default_us  HOST or NULL: median step time under the pinned order / under the planner's own
 * A step with no decodes or no chunk has one grid and nothing to order (returns at once).  Errors as kairos_mixed_step.
 */
int kairos_tune_step(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                     int32_t dec_table_stride, const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len,
                     const void* q_chunk, const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec,
                     void* out_chunk, int32_t reps, int32_t* chosen_mode, double* chosen_us, double* default_us,
                     void* cuda_stream);

/*
 * the fp8 latent cache ("an fp8 latent-cache variant (halves the decode roofline)").  The paper has no
 * such passage; the format is DESIGN.md reading G23:
 *   one cached token = 512 latent values as e4m3 codes (OCP fp8: bias 7, no infinity, largest finite 448) + ONE float32 scale
 *   + its 64 RoPE key values in bf16 = 644 bytes (bf16 cache: 1,152).  A page of 64 tokens is KAIROS_FP8_PAGE_BYTES = 41,216
 *   bytes:  codes u8 [64][512]  |  RoPE bf16 [64][64] at byte 32,768  |  scales f32 [64] at byte 40,960.
 *   Quantisation of token t (float32, IEEE round to nearest even): amax = max_d |c_t[d]|;  s_t = amax / 448 (1 when amax = 0);
 *   code = e4m3_rne_satfinite(c_t[d] / s_t).  The cached latent is s_t * value(code); attention is the definition at the top of
 *   this file over those values (q in bf16, fp32 accumulation, bf16 out).  Inside the kernel the MMAs are tcgen05 kind::f8f6f4
 *   on the codes themselves; q and the softmax weights enter them as a sum of two e4m3 terms (a 4-bit head and the 4-bit
 *   remainder), which keeps them at bf16's precision -- see DESIGN.md 6.7 for the error budget.
 *
 * kairos_fp8_attach     tells the context about an fp8 pool: pool8 DEVICE [num_pages][41,216] bytes, 128-byte aligned.  It stays
 *                       caller-owned and must outlive the context or the next attach.  The bf16 pool given at create time is
 *                       untouched: a context can serve both.
 * kairos_fp8_append     as kairos_append_latent (same arguments, same indexing, same errors) but quantises into the attached
 *                       fp8 pool.  BIT-EXACT against the definition above: codes, scales and RoPE bytes.
 * kairos_fp8_append_decode_tokens  as kairos_append_decode_tokens: request i caches its newest token at positions[i] through row i of
 *                       page_tables (quantised as above; positions are trusted, device-side only).
 * kairos_fp8_decode     as kairos_mixed_step with chunk_len = 0 over the fp8 pool: n_dec decodes, request i attends its first
 *                       dec_ctx_lens[i] cached tokens through row i of dec_page_tables.  Same planner (a0), split partials,
 *                       LSE combine, plan cache and graph replay as the bf16 step; q is split into its two e4m3 terms inside
 *                       the kernel (no extra launch, no scratch).  Stale slots of a request's last page never reach a result
 *                       (any bit pattern, NaN codes included).
 * kairos_fp8_mixed_step the mixed step itself over the fp8 pool (same arguments as kairos_mixed_step; the chunk's tokens must already be
 *                       in the cache: kairos_fp8_append at start_pos = prefix_len).  There is no fp8 chunk-tile kernel: token j of
 *                       the chunk runs as a one-token request over the chunk's own sequence (n_keys = prefix_len + j + 1) in the same
 *                       grid as the decodes, its pages kept in L2 (evict-last) for the later tokens.  That serves the chunk sizes
 *                       the paper deflects with (chi = 128 .. 2048 beside a decode batch); a long chunk over a
 *                       long prefix re-reads the prefix once per token and belongs on the bf16 path's cluster kernel.  The
 *                       workspace must cover max_decodes + max_chunk requests: kairos_workspace_bytes(max_decodes + max_chunk, 0).
 * Errors: INVALID_ARG (NULL / misaligned / sizes / no pool attached), WORKSPACE, CUDA.
 */
#define KAIROS_FP8_PAGE_BYTES 41216
int kairos_fp8_attach(kairos_ctx* ctx, void* pool8, int32_t num_pages);
int kairos_fp8_append(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n_tokens, const int32_t* page_table,
                      int32_t table_len, int32_t start_pos, void* cuda_stream);
int kairos_fp8_append_decode_tokens(kairos_ctx* ctx, const void* latent, const void* k_rope, int32_t n, const int32_t* page_tables,
                                    int32_t table_stride, const int32_t* positions, void* cuda_stream);
int kairos_fp8_mixed_step(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                          const int32_t* dec_ctx_lens, int32_t chunk_len, int32_t prefix_len, const void* q_chunk,
                          const int32_t* chunk_page_table, int32_t chunk_table_len, void* out_dec, void* out_chunk, float* lse_dec,
                          float* lse_chunk, void* cuda_stream);
int kairos_fp8_decode(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables,
                      int32_t dec_table_stride, const int32_t* dec_ctx_lens, void* out_dec, float* lse_dec, void* cuda_stream);

/*
 * Decode attention for callers that MAY NOT ALLOCATE (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc).  kairos_mixed_step grows pinned and device plan buffers on demand and takes its split-KV scratch from the caller's
 * workspace; this entry point does neither: the queue counters, the work list, the combine list and the fp32 split partials live in
 * ONE fixed array of device memory that is part of the library image (`static __device__`, about 9.3 MiB; every GPU that loads
 * libkairos.so holds it until the process exits), and the work list is written by a small kernel on the device.  The call makes
 * three launches (plan, decode splits, LSE combine) and no cudaMalloc / cudaFree / allocating library call.
 *   Same operation and argument meaning as kairos_mixed_step with chunk_len = 0: request i attends its first dec_ctx_lens[i] cached
 *   tokens of the bf16 pool through row i of dec_page_tables; out_dec bf16 [n_dec][16][512], lse_dec fp32 [n_dec][16] or NULL.
 *   Results agree with kairos_mixed_step within the attention tolerance (the KV split points differ, so not bit for bit).
 * Limits: n_dec <= KAIROS_STATIC_MAX_DECODES (128); any context length the page tables cover.  More decodes: KAIROS_ERR_WORKSPACE
 * with a message that names the limit -- use kairos_mixed_step.
 * Sharing: every call on a device, from every context, uses the SAME array, and the array keeps the last call's contents.  Each
 * call clears the counters and rewrites both lists before it reads them, so back-to-back calls on one stream are safe; calls that
 * overlap on the GPU (two streams, two contexts, two threads) race and corrupt each other -- serialise them.
 * Asynchronous on `cuda_stream`; dec_ctx_lens (HOST) is read before the call returns.  Errors: INVALID_ARG, WORKSPACE, CUDA.
 */
#define KAIROS_STATIC_MAX_DECODES 128
int kairos_decode_static(kairos_ctx* ctx, int32_t n_dec, const void* q_dec, const int32_t* dec_page_tables, int32_t dec_table_stride,
                         const int32_t* dec_ctx_lens, void* out_dec, float* lse_dec, void* cuda_stream);

/*
 * TEST-ONLY knobs (parity tests force every launch order and code path through them; sweeps under profiles/ use them;
 * a deployment never calls this).  Takes effect from the next kairos_mixed_step.
 *   "pairs"       -1 planner decides (default); 0 never use the cluster kernel; n > 0 decode grid first beside n clusters;
 *                 -(n + 1) n clusters first, the decode grid behind them (see kairos_plan_dump pair_mode)
 *   "dec_only"    0 = never use the decode-only instantiation of the queue kernel; -1 default
 *   "copy_stream" 0 = plan copies on the caller's stream; 1 default (the context's copy stream)
 *   "graph"       0 = never replay a plan as a CUDA graph; 1 default
 *   "plan_cache"  0 = plan every step; 1 default
 *   "host_slice_tokens"  kairos_mixed_step_host: n > 0 = slices of n chunk tokens (rounded up to whole 8-token tiles); 0 default (its own rule)
 * Errors: INVALID_ARG for an unknown key.
 */
int kairos_debug_set(kairos_ctx* ctx, const char* key, int32_t value);

/* Message for the last failing call on this thread ("" if none; thread-local, so no context argument). Never NULL. */
const char* kairos_last_error(void);

/* Library build tag, e.g. "kairos-b200 sm_100a <kernel generation>". Never NULL. */
const char* kairos_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KAIROS_H_ */
