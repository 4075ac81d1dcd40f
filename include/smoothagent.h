/*
 * smoothagent.h -- C ABI of the B200-native re-prefill hot path of SmoothAgent
 * (arxiv/paper_2607_00151, "lookahead context engineering").
 *
 * What the path computes (PAPER.md = the paper text, line numbers Lnnn):
 *   After a context transformation the transformed segment must be re-prefilled: its K/V are
 *   built and its tokens attend causally to the retained prefix held in a paged KV cache plus
 *   themselves (L37, L105-109, L168).  Lookahead re-prefill chunks are co-batched with
 *   latency-critical decode rows (L392-398).  Per request j the batch carries q_j new query
 *   tokens over prefix_j cached tokens; "the i-th query token attends to prefix_j + i + 1
 *   tokens" (L311-313); a decode request is "a single query token that attends to its full KV
 *   cache of length L_j" (L305).  The scheduler's latency model (Eq. 1) consumes
 *   profiled attention costs: sa_latency_table measures them.
 *
 * Conventions
 *   - Every call returns an int32_t status: SA_OK or a negative SA_ERR_*.  No exceptions, no
 *     exit(), nothing is printed.  sa_status_string() names a status.
 *   - "device" pointers are CUDA device pointers on the pool's device; "host" pointers are
 *     ordinary host memory.  THE CALLER OWNS EVERY DEVICE BUFFER (pool storage, q/k/v inputs,
 *     outputs, workspace); the library owns host metadata only.  Host arrays passed to a call
 *     are copied before it returns and may be reused at once.
 *   - Hot calls (sa_rope_kv_append, sa_mixed_attention) take a CUDA stream as void*
 *     (cudaStream_t; NULL = the legacy default stream), only enqueue work, never allocate
 *     device memory and never synchronise the device.  All hot calls on one pool must be
 *     issued on one stream (or on streams the caller orders).  A pool is not thread-safe.
 *     They may wait on the host for a metadata slot of an earlier call and change host-side
 *     session state when called, so they must not be issued under CUDA stream capture; the capturable form of a
 *     decode iteration is sa_decode_step_prepare (host) + sa_decode_step_enqueue (device).
 *   - A call that fails with SA_ERR_INVALID_ARG, SA_ERR_OUT_OF_PAGES, SA_ERR_OUT_OF_SESSIONS, SA_ERR_UNSUPPORTED or
 *     SA_ERR_WORKSPACE_TOO_SMALL leaves the pool, its block tables and session lengths unchanged: everything is
 *     validated and sized before any state is touched.  SA_ERR_CUDA means the CUDA runtime refused a launch, copy or
 *     event (in practice a sticky device error from earlier work): host bookkeeping may by then have moved on (pages
 *     taken, sessions grown or committed, part of a layer enqueued), so the pool's state is undefined and the only
 *     valid call on it is sa_kv_pool_destroy.
 *   - Every call that touches the device runs on the pool's device (cfg.device) whatever device is current in the
 *     calling thread, and restores the caller's current device before returning.  The pool-less dense operators
 *     (sa_linear, sa_swiglu, sa_rmsnorm, sa_gemm_table) run on the current device.
 *   - All tensors are bf16 (raw 16-bit patterns), packed ragged: the tokens of request r are
 *     rows [qo_indptr[r], qo_indptr[r+1]) of a [T, heads, head_dim] row-major array.
 *   - There is no CPU fallback: without a CUDA device the hot calls return SA_ERR_CUDA.
 *
 * Supported shapes: head_dim in {64, 128}; page_size in {16, 64}; num_q_heads a multiple of
 * num_kv_heads with group size G = Hq/Hkv in {1, 2, 4, 8, 16}.  Anything else:
 * SA_ERR_UNSUPPORTED.
 */
#ifndef SMOOTHAGENT_H_
#define SMOOTHAGENT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define SA_API __attribute__((visibility("default")))
#else
#define SA_API
#endif

#define SA_OK 0
#define SA_ERR_INVALID_ARG (-1)
#define SA_ERR_OUT_OF_PAGES (-2)
#define SA_ERR_UNSUPPORTED (-3)
#define SA_ERR_CUDA (-4)
#define SA_ERR_WORKSPACE_TOO_SMALL (-5)
#define SA_ERR_OUT_OF_SESSIONS (-6)

typedef struct sa_kv_pool sa_kv_pool; /* opaque */

typedef struct {
    int32_t num_q_heads;        /* Hq */
    int32_t num_kv_heads;       /* Hkv; q head h reads kv head h / (Hq/Hkv)  (GQA, L422) */
    int32_t head_dim;           /* D */
    int32_t page_size;          /* B: tokens per page */
    int64_t num_pages;          /* pages in the pool */
    int32_t max_sessions;       /* concurrently open sessions */
    int32_t device;             /* CUDA device ordinal of dev_storage */
    int64_t max_session_tokens; /* longest context one session may reach (sizes its block table) */
    double rope_base;           /* theta_m = rope_base^(-2m/D); half-split pairing (m, m + D/2) */
} sa_kv_pool_config;

/* Where a slot lives, so a caller (or a test) can address any K/V element:
 *   element (page p, kv head g, slot s, dim d) of K is  k_base[p*stride_page + g*stride_head
 *   + s*stride_slot + d]  (strides in bf16 elements, d contiguous); same for v_base. */
typedef struct {
    void *k_base;
    void *v_base;
    int64_t stride_page;
    int64_t stride_head;
    int64_t stride_slot;
} sa_kv_layout;

SA_API const char *sa_status_string(int32_t status);

/* ---- sa_kv_pool_create: the page pool and block tables -------------
 * Bytes of device storage a pool of this configuration needs (K pages, V pages, the device
 * mirror of the block tables, RoPE frequency table, per-call metadata ring). */
SA_API int32_t sa_kv_pool_storage_bytes(const sa_kv_pool_config *cfg, size_t *out_bytes);

/* Create a pool over caller-owned device storage (256-byte aligned, >= storage_bytes).
 * free_page_order (host, nullable): a permutation of [0, num_pages); pages are handed out in
 * this order (NULL = 0,1,2,...), which is how tests pick the physical page map.
 * dev_storage == NULL creates a HOST-ONLY pool: session and page bookkeeping work (including
 * the page allocation of sa_rope_kv_append, which then moves no data), sa_mixed_attention and
 * sa_latency_table return SA_ERR_CUDA.  Used by the CPU tests of the allocator and planner.
 * The storage is not cleared: page contents are whatever the caller left there. */
SA_API int32_t sa_kv_pool_create(const sa_kv_pool_config *cfg, void *dev_storage, size_t bytes,
                          const int32_t *free_page_order, sa_kv_pool **out_pool);
SA_API int32_t sa_kv_pool_destroy(sa_kv_pool *pool);
SA_API int32_t sa_kv_pool_layout(const sa_kv_pool *pool, sa_kv_layout *out);
SA_API int32_t sa_kv_pool_free_pages(const sa_kv_pool *pool, int64_t *out_free_pages);

/* Sessions: one logical context = an ordered list of pages + a length in tokens. */
SA_API int32_t sa_kv_session_open(sa_kv_pool *pool, int32_t *out_sid);
SA_API int32_t sa_kv_session_close(sa_kv_pool *pool, int32_t sid); /* returns its pages to the pool */
/* Keep the retained prefix [0, new_len), drop the invalidated tail (the context transformation
 * "invalidates the existing KV cache" from the first changed token on, L37).  Pages wholly
 * beyond new_len go back to the free list (most recently freed is reused first). */
SA_API int32_t sa_kv_session_truncate(sa_kv_pool *pool, int32_t sid, int64_t new_len);
/* len (nullable): tokens; pages (nullable, host): receives min(*n_pages, used) page ids;
 * n_pages (nullable, in/out): capacity in, pages used out. */
SA_API int32_t sa_kv_session_query(const sa_kv_pool *pool, int32_t sid, int64_t *len, int32_t *pages,
                            int32_t *n_pages);

/* ---- session operations of the commit splice ------------------------------
 * A lookahead request rebuilds the transformed context's KV ahead of time in a session of its own
 * and, at the commit point, "directly replaces the prefix in the working context" (L47, L170,
 * L186-187); sub-agent contexts are built chunk by chunk while the main agent decodes (L265-281).
 *
 * sa_kv_session_fork: open a new session whose first prefix_len tokens are those of src_sid (the
 * retained prefix).  Whole pages of the prefix are SHARED (reference-counted, never written
 * again); if the prefix ends inside a page, that page is copied into a fresh page now (enqueued
 * on `stream`), so the two sessions append independently.  Needs at most one free page.
 * sa_rope_kv_append also copies on write: appending into a partly filled last page that another
 * session still holds first moves the appender to a private copy of that page.
 * sa_kv_session_commit: main_sid takes over the lookahead session's pages and length (its device
 * block-table row is rewritten on `stream`), the pages it held before lose a holder, and
 * lookahead_sid is closed.  A page returns to the free list when its last holder lets go. */
SA_API int32_t sa_kv_session_fork(sa_kv_pool *pool, int32_t src_sid, int64_t prefix_len, int32_t *out_sid,
                           void *stream);
SA_API int32_t sa_kv_session_commit(sa_kv_pool *pool, int32_t main_sid, int32_t lookahead_sid, void *stream);
SA_API int32_t sa_kv_page_refcount(const sa_kv_pool *pool, int32_t page, int32_t *out_refs);

/* ---- sa_rope_kv_append: fused RoPE + scatter of new K/V into pages (step a2) -------------
 * Request r appends q_r = qo_indptr[r+1]-qo_indptr[r] tokens to session sids[r]; token i of
 * request r sits at absolute position session_len(r) + i IN THE TRANSFORMED CONTEXT (the
 * segment starts right after the retained prefix, L105-109).  K is rotated at that position
 * (computed in fp32 with a split-precision angle, one round-to-nearest-even to bf16) and
 * stored; V is copied bit for bit; q_inout (nullable) is rotated in place at the same
 * positions.  Pages are allocated as needed; on SA_ERR_OUT_OF_PAGES nothing is changed.
 * A session may appear at most once per call.  Slots not addressed by the call keep their bits.
 *   sids, qo_indptr : host, n_req and n_req+1 entries, qo_indptr[0] == 0, non-decreasing
 *   k, v            : device bf16 [T, Hkv, D], pre-RoPE
 *   q_inout         : device bf16 [T, Hq, D], nullable */
SA_API int32_t sa_rope_kv_append(sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                          const int32_t *qo_indptr, const void *k, const void *v, void *q_inout,
                          void *stream);

/* ---- sa_mixed_attention: ragged batch of prefill chunks and decode rows (steps a3-a6) -----
 * Request r has q_r query rows and attends to its session's cache of kv_r = session_len(r)
 * tokens, WHICH ALREADY CONTAINS its own q_r tokens (append first, then attend; L305 "its full
 * KV cache").  Row i of request r attends keys 0 .. kv_r - q_r + i (L311-313), softmax in fp32
 * with scale sm_scale, GQA head mapping h -> h / G.  q_r == 1 is a decode row, q_r > 1 a
 * prefill chunk, q_r == 0 a no-op; they may be mixed freely in one call.  The bits of a decode
 * row's output depend only on that request; the bits of a prefill row depend on the set of
 * prefill requests of the call (their work is balanced over the SMs by cutting items along KV,
 * see sa_mixed_attention_schedule) and not on the decode rows co-batched with them; neither depends
 * on which physical pages hold the cache.  Contents of page slots >= kv_r never influence a result, NaN included.
 * The call only reads the cache, so a session may be named by several requests of one call; each request is then what
 * it would be alone (its rows are the last q_r tokens of that session).  sa_rope_kv_append, which writes, refuses that.
 *   q    : device bf16 [T, Hq, D], already rotated (sa_rope_kv_append's q_inout)
 *   out  : device bf16 [T, Hq, D]
 *   lse  : device f32 [T, Hq], nullable; natural-log sum-exp of the scaled scores of the row
 *   sm_scale <= 0 selects 1/sqrt(D)
 *   workspace : device, >= sa_mixed_attention_workspace_bytes(...) for the same batch */
SA_API int32_t sa_mixed_attention_workspace_bytes(const sa_kv_pool *pool, int32_t n_req,
                                           const int32_t *sids, const int32_t *qo_indptr,
                                           size_t *out_bytes);
SA_API int32_t sa_mixed_attention(sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                           const int32_t *qo_indptr, const void *q, void *out, float *lse,
                           float sm_scale, void *workspace, size_t workspace_bytes, void *stream);

/* The three planning calls below take a `const sa_kv_pool *` because they change nothing a caller can observe, but
 * they do write a per-pool cache (the plan of the last batch planned, which the sa_mixed_attention call that follows
 * takes over instead of planning again) and sa_mixed_attention_schedule / _plan read it.  Like every call on a pool
 * they must therefore be serialised with the other calls on that pool: a scheduler thread sizing a batch while a worker
 * thread enqueues on the same pool is a data race.  Plan on a host-only twin pool if two threads must do both.
 *
 * Host-side planner statistics of the batch sa_mixed_attention would run (no device work; works
 * on host-only pools).  out_stats (host int64[8]) = { decode-like requests, prefill requests,
 * decode CTAs, prefill work items (parts of the schedule on the tcgen05 path), split partial rows, sum_j L_j over decode-like requests,
 * sum_j A_j over prefill requests (A_j = q_j*prefix_j + q_j(q_j+1)/2, L313), 1 if prefill chunks
 * run on the tcgen05 kernel (always, for the supported shapes) }. */
SA_API int32_t sa_mixed_attention_plan(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                const int32_t *qo_indptr, int64_t *out_stats);

/* The static schedule the tcgen05 prefill kernel would run for this batch (host only; works on
 * host-only pools; every supported shape takes the tcgen05 path).  An item is
 * (request, kv head, tile of 256 packed rows: row rho = token*G + head-in-group); its cost is n_kv =
 * the number of 128-key tiles it attends to (the causal work A_j of L313 in tiles).  Items are
 * assigned to one persistent CTA per SM; an item that does not fit under the balanced makespan is
 * cut along KV into parts [u0, u1) whose partial results are merged in KV order.
 *   out_parts (host int32 [cap][8], nullable): per part {cta, request index in the caller's list,
 *       kv head, tile, u0, u1, n_kv, partial slot or -1 for a whole item}, grouped by CTA in
 *       execution order; at most cap rows are written
 *   out_summary (host int64 [6]): {CTAs, parts, split items, partial slots, sum of n_kv over
 *       items, largest CTA load in tiles incl. the fixed cost per part} */
SA_API int32_t sa_mixed_attention_schedule(const sa_kv_pool *pool, int32_t n_req, const int32_t *sids,
                                    const int32_t *qo_indptr, int32_t *out_parts, int32_t cap,
                                    int64_t *out_summary);

/* ---- sa_decode_step_*: one decode iteration, capturable in a CUDA graph (steps a1-a2, a5-a6) -----------------------
 * The latency-critical class of the runtime is the decode iteration (its time is the TBT that
 * Algorithm 2 protects, L392-398): every request appends ONE token and its query row attends to the whole cache, own
 * token included.  sa_rope_kv_append + sa_mixed_attention compute that, but plan on the host inside the call, so
 * they cannot be recorded once and replayed.  A decode step separates the two halves:
 *   sa_decode_step_prepare   HOST ONLY (no device work, nothing enqueued).  For each request: the host half of
 *       appending one token to sids[r] (a page is taken when the session's last page is full; the session grows by
 *       one) and the attention plan of its row.  Everything the kernels need is written to a pinned slab the step
 *       owns.  Must not be called while an earlier enqueue / graph replay of this step can still be running (the
 *       kernels read the slab when they execute).  Errors leave the pool and the step unchanged: SA_ERR_INVALID_ARG
 *       (n_req > max_requests, unknown / closed / repeated session, cache would exceed max_kv_tokens),
 *       SA_ERR_OUT_OF_PAGES, SA_ERR_UNSUPPORTED (a session whose partly filled last page is shared with a fork: the
 *       copy-on-write needs sa_rope_kv_append).
 *   sa_decode_step_enqueue   DEVICE ONLY.  Enqueues two launches with fixed grids on `stream` and changes no host
 *       state: (1) slab -> device twin, RoPE + placement of the new tokens (K rotated at the token's position, V bit
 *       copy, q_inout rotated in place, block-table entry written), (2) split-KV attention of the rows, the actual
 *       counts read on the device, the last split of a row merging them.  Legal under CUDA stream capture; the captured graph is
 *       replayed after each prepare (same k / v / q_inout / out / lse addresses, new contents).  Calling it again
 *       without a new prepare re-places the same tokens and recomputes the same rows, provided q_inout holds the RAW
 *       rows again (it is rotated in place each time the kernels run).
 * Results are bit-equal to sa_rope_kv_append + sa_mixed_attention on the same batch (same device code per row).
 *   max_requests   : capacity of a step (<= cfg.max_sessions); max_kv_tokens: longest cache a row may attend to
 *   dev_mem        : device, 256-byte aligned, >= sa_decode_step_device_bytes(...): metadata twin + split partials;
 *                    the caller's, and must outlive the step (NULL for a host-only pool)
 *   k, v           : device bf16 [n_req, Hkv, D], pre-RoPE; q_inout: device bf16 [n_req, Hq, D]
 *   out            : device bf16 [n_req, Hq, D]; lse: device f32 [n_req, Hq], nullable
 *   sa_decode_step_stats: host int64[6] = {requests, work items, CTAs of the attention grid, launches of the last
 *                    enqueue, partial rows the workspace holds, capacity}
 * One prepare, one execution.  Every successful prepare must be followed by an execution of the step -- an
 * sa_decode_step_enqueue, or a replay of the graph it was captured into -- before the next prepare.  The library cannot see
 * graph replays, so it cannot check this; a prepare that is never executed leaves its sessions one token longer with
 * nothing written at that position (and, where it took a page, a device block-table entry that stays unwritten until a
 * later step places a token in that page), and a later attention over such a session reads whatever those slots held.
 *   sa_decode_step_cancel    HOST ONLY.  Undoes the step's last successful prepare when it will not be executed (the batch
 *       changed, a request was aborted): the sessions get their old lengths back, pages the prepare took return to the
 *       free list so that they are handed out again in the same order, and the step holds no batch (enqueue is refused
 *       until the next prepare; a replay of an already captured graph does nothing).  SA_ERR_INVALID_ARG, with nothing
 *       changed, if there is no prepare to undo (none yet, or already cancelled) or one of its sessions has been closed,
 *       grown or truncated since.  Cancelling a prepare that HAS executed amounts to truncating its sessions by one token.
 * Lifetime: a step refers to its pool in every call except sa_decode_step_destroy; destroy the steps of a pool before
 * the pool, or at least never prepare / enqueue / cancel / query a step once its pool is gone. */
typedef struct sa_decode_step sa_decode_step; /* opaque */
SA_API int32_t sa_decode_step_device_bytes(const sa_kv_pool *pool, int32_t max_requests, int64_t max_kv_tokens,
                                           size_t *out_bytes);
SA_API int32_t sa_decode_step_create(sa_kv_pool *pool, int32_t max_requests, int64_t max_kv_tokens, void *dev_mem,
                                     size_t dev_bytes, sa_decode_step **out_step);
SA_API int32_t sa_decode_step_destroy(sa_decode_step *step);
SA_API int32_t sa_decode_step_prepare(sa_decode_step *step, int32_t n_req, const int32_t *sids);
SA_API int32_t sa_decode_step_cancel(sa_decode_step *step);
SA_API int32_t sa_decode_step_enqueue(sa_decode_step *step, const void *k, const void *v, void *q_inout, void *out,
                                      float *lse, float sm_scale, void *stream);
SA_API int32_t sa_decode_step_stats(const sa_decode_step *step, int64_t *out_stats);

/* Number of kernel launches the last successful sa_mixed_attention / sa_rope_kv_append on this
 * pool enqueued (for launch accounting in benchmarks). */
SA_API int32_t sa_last_launch_count(const sa_kv_pool *pool, int32_t *out_launches);

/* ---- sa_latency_table: device-level latency model input (step a7) -------------------------
 * Measures the time of one sa_mixed_attention call for every (prefill_tokens[a],
 * decode_batch[b]) pair: the profiled attention terms of Eq. 1 (L305-319, L349-353; "offline-
 * profiled", L303).  Prefill tokens p are issued as ceil(p/2048) chunks of <= 2048 tokens, each
 * over its own prefix of prefill_prefix_len tokens; decode rows have contexts drawn uniformly
 * from [decode_ctx_lo, decode_ctx_hi] with a counter-based generator seeded by seed.
 * NOT a hot call: it opens scratch sessions in the pool's free pages (at most max(decode_batch) + ceil(max(prefill_tokens)
 * / 2048) of them: SA_ERR_OUT_OF_SESSIONS / SA_ERR_OUT_OF_PAGES before anything is opened), synchronises the stream, and
 * closes the sessions before returning.  It allocates no device memory: its source K/V, queries, outputs, the 256 MiB buffer
 * it writes between timed iterations to evict L2 and the attention workspace all come from `workspace`
 * (>= sa_latency_table_workspace_bytes for the same arguments; that call replays the run's sessions on a host-only twin of
 * the pool, so the figure is the planner's own).
 *   out_ms : host float [n_p][n_d], median over iters of CUDA-event times on `stream`
 *   out_sum_kv (nullable): host int64 [n_p][n_d][2] = {sum_j L_j of the decode rows,
 *                          sum_j A_j of the prefill chunks} for fitting alpha_d, alpha_p */
SA_API int32_t sa_latency_table_workspace_bytes(const sa_kv_pool *pool, const int32_t *prefill_tokens, int32_t n_p,
                                         const int32_t *decode_batch, int32_t n_d, int64_t prefill_prefix_len,
                                         int64_t decode_ctx_lo, int64_t decode_ctx_hi, uint64_t seed, size_t *out_bytes);
SA_API int32_t sa_latency_table(sa_kv_pool *pool, const int32_t *prefill_tokens, int32_t n_p,
                         const int32_t *decode_batch, int32_t n_d, int64_t prefill_prefix_len,
                         int64_t decode_ctx_lo, int64_t decode_ctx_hi, uint64_t seed,
                         int32_t warmup, int32_t iters, float *out_ms, int64_t *out_sum_kv,
                         void *workspace, size_t workspace_bytes, void *stream);

/* ---- lookahead-aware scheduler core (section 4) --------------
 * Host-only calls (no device work, no pool): the consumer of sa_latency_table.
 *
 * Latency model (Eq. 1):
 *     EstBatchLatency(B) = c0 + T_GEMM(M) + alpha_d * sum_{j in decode} L_j + alpha_p * sum_{j in prefill} A_j
 * M = |B_decode| + sum_j q_j (L301); L_j = cache length of decode request j (L305); A_j = q_j*prefix_j +
 * q_j(q_j+1)/2 (L313).  c0 is a fixed cost per call that the paper's equation does not have (0
 * reproduces it).  T_GEMM(M): the offline-profiled lookup table with interpolation of L299-303,
 * piecewise linear through (gemm_m[i], gemm_ms[i]), constant below the first point, the last
 * segment's slope beyond the last; n_gemm = 0 gives T_GEMM = 0 (this path has no GEMMs).  An empty
 * batch costs 0.  Estimates are computed in double, the three integer sums exactly. */
#define SA_GEMM_TABLE_MAX 64
typedef struct {
    double c0_ms;
    double alpha_d_ms;                  /* ms per cached token read by decode rows */
    double alpha_p_ms;                  /* ms per causal (query, key) pair of prefill chunks */
    int32_t n_gemm;
    int32_t reserved;
    double gemm_m[SA_GEMM_TABLE_MAX];   /* strictly increasing */
    double gemm_ms[SA_GEMM_TABLE_MAX];
} sa_latency_model;

typedef struct {
    int64_t q;      /* query tokens of the chunk (q_j) */
    int64_t prefix; /* cached tokens before them (prefix_j) */
} sa_chunk;

typedef struct {
    double t_arrival_ms;
    double slo_ttft_ms;
    int64_t q;      /* prefill tokens the request still needs */
    int64_t prefix; /* tokens of it already cached */
} sa_lc_request;

/* Least-squares fit of ms[i] ~ c0 + alpha_d*sum_kv[i][0] + alpha_p*sum_kv[i][1] over n profiled batches:
 * exactly the out_ms / out_sum_kv arrays of sa_latency_table ("profiled coefficient", L309, L319).
 * with_intercept == 0 fits Eq. 1 literally (c0 = 0).  A column that is zero in every batch keeps a zero
 * coefficient.  out_max_rel_err (nullable): max_i |fit_i - ms_i| / ms_i.  out->n_gemm is set to 0. */
SA_API int32_t sa_latency_fit(const float *ms, const int64_t *sum_kv, int32_t n, int32_t with_intercept,
                       sa_latency_model *out, double *out_max_rel_err);

SA_API int32_t sa_est_batch_latency(const sa_latency_model *model, const int64_t *decode_L, int32_t n_dec,
                             const sa_chunk *chunks, int32_t n_pre, double *out_ms);

/* Algorithm 2 (PD co-located, L363-388): admit decode requests, then LC prefill chunks, then BE
 * (lookahead) chunks, each queue in order, each candidate only while EstBatchLatency(B + {c}) <=
 * delta_ms; the first candidate of a queue that does not fit ends that queue.
 * out_admitted (host int32[3]) = admitted {decode, LC chunks, BE chunks}: always a prefix of each queue.
 * out_est_ms (nullable): the estimate of the admitted batch. */
SA_API int32_t sa_schedule_hybrid(const sa_latency_model *model, const int64_t *decode_L, int32_t n_dec,
                           const sa_chunk *lc, int32_t n_lc, const sa_chunk *be, int32_t n_be,
                           double delta_ms, int32_t *out_admitted, double *out_est_ms);

/* Algorithm 1 (PD disaggregated, L321-347): lc_queue is the LC queue in the order of the LC policy;
 * p accumulates EstPrefillLatency(r) (= Eq. 1 of r's remaining prefill alone), the slack of request j is
 * (t_arrival + SLO_TTFT) - t_now - p, t_budget = max(0, min_j slack) (+inf with an empty queue).
 * lc_chunks = NextChunks(Q_LC) is always in the batch; BE chunks are admitted in order while
 * EstBatchLatency(B_LC + B_BE + {c}) <= t_budget, and the first one that does not fit ends the scan
 * (the listing's lines 15-17 are garbled in PAPER.md; this is Algorithm 2's rule and keeps the
 * lookahead queue in order, L168). */
SA_API int32_t sa_schedule_prefill_slack(const sa_latency_model *model, const sa_lc_request *lc_queue, int32_t n_queue,
                                  double t_now_ms, const sa_chunk *lc_chunks, int32_t n_lc_chunks,
                                  const sa_chunk *be, int32_t n_be, int32_t *out_be_admitted,
                                  double *out_budget_ms, double *out_est_ms);

/* Dynamic chunking (L59, L359, L396): the largest next chunk of a lookahead prefill with `remaining`
 * tokens over `prefix` cached ones that keeps the batch (decode_L, chunks) within budget_ms:
 * min(remaining, max_chunk) if it fits, else the largest multiple of `granularity` below it that
 * fits, else 0. */
SA_API int32_t sa_dynamic_chunk(const sa_latency_model *model, const int64_t *decode_L, int32_t n_dec,
                         const sa_chunk *chunks, int32_t n_pre, int64_t prefix, int64_t remaining,
                         int64_t max_chunk, int64_t granularity, double budget_ms, int64_t *out_q);

/* ---- dense operators of the layer (section 4 "GEMM", L299-303) ----------
 * "All tokens in the batch, including decode tokens and prefill chunk tokens, are processed by the
 * same dense operators in each transformer layer, including the projection matrices in attention
 * (QKV and output projections) and the FFN layers" (L299); their cost T_GEMM(M) depends on the total
 * number of forward tokens M only (L301-303).  The layer is BASELINE.json's "Llama-3-8B-shaped"
 * pre-norm decoder layer without biases (readings R21-R24 in DESIGN.md):
 *     h  = RMSNorm(x; norm1)            q|k|v = h W_qkv^T  (rows of W_qkv: Hq Q heads, Hkv K heads, Hkv V heads)
 *     a  = attention(RoPE(q), RoPE(k), v)                   (sa_mixed_attention over the paged cache)
 *     x1 = x + a W_o^T
 *     h2 = RMSNorm(x1; norm2)
 *     y  = x1 + (SiLU(h2 W_gate^T) * (h2 W_up^T)) W_down^T
 * All tensors are device bf16, row-major, weights stored [out_features, in_features] (y = x W^T);
 * accumulation is fp32 on the tensor cores (tcgen05, TMEM accumulators), every stored tensor is
 * rounded once to bf16 (round to nearest even).  All calls enqueue on `stream`, never allocate and
 * never synchronise (sa_gemm_table excepted).  Shape limits of the tcgen05 GEMM: in_features a
 * multiple of 64, out_features a multiple of 8, every pointer 16-byte aligned, M >= 0 arbitrary.
 * Stream order: activations, residuals, outputs and workspaces are read and written in stream order.  WEIGHTS (w,
 * w_gate, w_up, w_qkv, the norm weights) are read AHEAD of it: the kernels are launched with programmatic stream
 * serialization and request their first weight tiles while the kernel before them in the stream may still be running
 * (they wait for it only before touching anything else).  A weight tensor must therefore not be written by work that
 * can still be in flight on the stream when the call is enqueued -- weights loaded once at start-up, the normal case,
 * are fine; a kernel that rewrites a weight matrix right before the call needs a synchronisation (or an event) first. */

/* y[M, N] = x[M, K] W[N, K]^T (+ residual[M, N] if non-null; y may alias residual). */
SA_API int32_t sa_linear(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N,
                  int32_t K, void *stream);

/* act[M, F] = SiLU(x W_gate^T) * (x W_up^T): one GEMM over both weight matrices with the activation fused
 * into its epilogue (the two products of an FFN unit are accumulated side by side in TMEM). */
SA_API int32_t sa_swiglu(const void *x, const void *w_gate, const void *w_up, void *act, int64_t M, int32_t F,
                  int32_t K, void *stream);

/* The same two operators with a scratch buffer.  With few rows (decode batches: the "near-constant latency"
 * regime of L301) the 128 x 256 tiles alone are too few to keep every SM streaming weights, so the K loop of a
 * tile is cut into slices that run on different SMs (split-K); fp32 partials go through `workspace` and a second
 * kernel sums them IN SLICE ORDER and applies the epilogue, so the result is bit-reproducible run to run (it may
 * differ in the last bit from the unsplit call: another summation order).  *_workspace_bytes returns 0 when the
 * shape will not be split; a null or too small workspace falls back to the unsplit kernel, never to an error -- so the
 * last bit of a result depends on whether the workspace was large enough: pass the same (sufficient) size every time
 * where bit-reproducibility across calls matters.  sa_qkv_rope_append and sa_layer_forward refuse a workspace smaller
 * than their *_workspace_bytes, which includes this scratch, so their split never varies. */
SA_API int32_t sa_linear_workspace_bytes(int64_t M, int32_t N, int32_t K, size_t *out_bytes);
SA_API int32_t sa_linear_ws(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N, int32_t K,
                     void *workspace, size_t workspace_bytes, void *stream);
SA_API int32_t sa_swiglu_workspace_bytes(int64_t M, int32_t F, int32_t K, size_t *out_bytes);
SA_API int32_t sa_swiglu_ws(const void *x, const void *w_gate, const void *w_up, void *act, int64_t M, int32_t F, int32_t K,
                     void *workspace, size_t workspace_bytes, void *stream);

/* sa_linear_noalloc: the split-K linear of sa_linear_ws for a caller that cannot provide `workspace`.
 * Every other call here leaves device memory to the caller, which is no help to a caller that has no allocator to
 * ask: an operator running inside an engine whose memory plan was fixed at start-up, a serving worker whose HBM has
 * all gone to the KV pool and the weights (a cudaMalloc of a few MiB then fails), a latency-critical loop that may
 * not call cudaMalloc / cudaFree because they can stall the whole device.  For those, the scratch of this one call
 * lives INSIDE THE LIBRARY: a fixed device array of SA_LINEAR_NOALLOC_SCRATCH_BYTES (20 MiB + 512 bytes) that the
 * driver sets aside on every GPU where this library's device code gets loaded and keeps until the process exits.
 * The call itself allocates and frees nothing, on the device or through any library routine; x, w, residual, y are
 * still the caller's (same meaning, layout and alignment rules as sa_linear; y may alias residual).
 *   Result    : the same kernels, split and summation order as sa_linear_ws with a full-size workspace -- bit-equal to it.
 *   Sizes     : only shapes the planner splits, i.e. sa_linear_workspace_bytes(M, N, K) != 0: few rows and a long K
 *               (ceil(M/128) * ceil(N/256) <= SMs/2 and K >= 256, e.g. M <= 512 at N = 4096 on 148 SMs).  Any other shape
 *               returns SA_ERR_UNSUPPORTED and touches nothing: it involves no scratch, so plain sa_linear already serves
 *               a caller that cannot allocate.  A shape whose scratch exceeds the array (possible only on a GPU with more
 *               than 160 SMs) returns SA_ERR_WORKSPACE_TOO_SMALL; the call never quietly runs unsplit.
 *   First call: the first call on each device looks the array's device address up (once per device and process, with
 *               the calling thread's current device; thread-safe).  That lookup may make the runtime load device code,
 *               so make this first call during start-up, before any stream capture begins on that device.
 *   Sharing   : every call on a device uses the same array and leaves its partial sums behind.  Nothing in it needs to
 *               be zero beforehand (each call writes every word it later reads), so stale contents are harmless, but
 *               two calls that can run on the GPU at the same time -- different streams without an event between them,
 *               or two host threads -- overwrite each other's partials and both results are garbage.  Issue them on one
 *               stream, or order them yourself.  Weights are read ahead of stream order as described above. */
#define SA_LINEAR_NOALLOC_SCRATCH_BYTES ((size_t)160 * 128 * 256 * 4 + 512)
SA_API int32_t sa_linear_noalloc(const void *x, const void *w, const void *residual, void *y, int64_t M, int32_t N,
                          int32_t K, void *stream);

/* y[M, H] = x / sqrt(mean_j x_j^2 + eps) * w  (fp32 arithmetic, one rounding). */
SA_API int32_t sa_rmsnorm(const void *x, const void *w, float eps, void *y, int64_t M, int32_t H, void *stream);

/* Fused QKV projection + RoPE + KV append: the same effect as projecting h with W_qkv and handing the
 * result to sa_rope_kv_append, but K', V go from the fp32 accumulators straight into the pool pages
 * and Q' into q_out, each rounded once (the unfused route rounds q, k twice).  Requests, positions,
 * page allocation, copy-on-write and failure behaviour are exactly sa_rope_kv_append's.
 *   h      : device bf16 [T, hidden]  (the normalised hidden states of the batch's new tokens)
 *   w_qkv  : device bf16 [(Hq + 2 Hkv) * D, hidden]
 *   q_out  : device bf16 [T, Hq, D], rotated queries for sa_mixed_attention
 *   workspace : device, >= sa_qkv_rope_append_workspace_bytes(T) (per-token cos/sin and slot table, plus the
 *               split-K scratch of a small batch)
 * Only head_dim 128 (SA_ERR_UNSUPPORTED otherwise). */
SA_API int32_t sa_qkv_rope_append_workspace_bytes(const sa_kv_pool *pool, int64_t total_tokens, size_t *out_bytes);
SA_API int32_t sa_qkv_rope_append(sa_kv_pool *pool, int32_t n_req, const int32_t *sids, const int32_t *qo_indptr,
                           const void *h, const void *w_qkv, int32_t hidden, void *q_out, void *workspace,
                           size_t workspace_bytes, void *stream);

typedef struct {
    int32_t hidden;      /* H */
    int32_t ffn;         /* F */
    float rms_eps;
    int32_t reserved;
    const void *norm1;   /* device bf16 [H] */
    const void *w_qkv;   /* device bf16 [(Hq + 2 Hkv) * D, H] */
    const void *w_o;     /* device bf16 [H, Hq * D] */
    const void *norm2;   /* device bf16 [H] */
    const void *w_gate;  /* device bf16 [F, H] */
    const void *w_up;    /* device bf16 [F, H] */
    const void *w_down;  /* device bf16 [H, F] */
} sa_layer_weights;

/* One decoder layer over a mixed batch (the formulas above): RMSNorm, fused QKV + RoPE + append,
 * sa_mixed_attention, output projection + residual, RMSNorm, SwiGLU GEMM, down projection + residual.
 * The batch is described as for sa_rope_kv_append (request r appends and queries q_r new tokens:
 * a prefill chunk if q_r > 1, a decode row if q_r == 1).
 *   x : device bf16 [T, H] in;  y : device bf16 [T, H] out (may alias x)
 *   workspace : device, >= sa_layer_workspace_bytes(...) for the same batch */
SA_API int32_t sa_layer_workspace_bytes(const sa_kv_pool *pool, const sa_layer_weights *layer, int32_t n_req,
                                 const int32_t *sids, const int32_t *qo_indptr, size_t *out_bytes);
SA_API int32_t sa_layer_forward(sa_kv_pool *pool, const sa_layer_weights *layer, int32_t n_req, const int32_t *sids,
                         const int32_t *qo_indptr, const void *x, void *y, float sm_scale, void *workspace,
                         size_t workspace_bytes, void *stream);

/* T_GEMM(M), the "offline-profiled lookup table" of L303: for every M in m_list the time of the layer's
 * dense operators on M tokens (QKV projection, output projection + residual, SwiGLU GEMM, down
 * projection + residual, the two RMSNorms), median over iters of CUDA-event times on `stream`, L2
 * evicted between iterations.  NOT a hot call (it synchronises), but it allocates nothing: weights and activations of the
 * given shape (values irrelevant to the timing), the L2-eviction buffer and the split-K scratch are carved from `workspace`
 * (device, >= sa_gemm_table_workspace_bytes for the same arguments; about 0.8 GB for the Llama-3-8B layer at M = 8192).
 * The result goes into sa_latency_model.gemm_m / gemm_ms. */
SA_API int32_t sa_gemm_table_workspace_bytes(int32_t hidden, int32_t ffn, int32_t num_q_heads, int32_t num_kv_heads,
                                      int32_t head_dim, const int32_t *m_list, int32_t n_m, size_t *out_bytes);
SA_API int32_t sa_gemm_table(int32_t hidden, int32_t ffn, int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                      const int32_t *m_list, int32_t n_m, int32_t warmup, int32_t iters, float *out_ms,
                      void *workspace, size_t workspace_bytes, void *stream);

/* ---- KV hand-over between pools ----------------------------------------------------
 * in PD-disaggregated serving "KV transfer" moves a request's cache from the prefill
 * instance to the decode instance (L456: 4 prefill + 4 decode GPUs); L424: tensor parallelism shards
 * the kv heads over GPUs.  A session's tokens travel as a WIRE IMAGE: dense bf16
 *     image[c][h][t][d],  c in {0: K' (rotated, as stored), 1: V},  h < Hkv,  t < n_tokens,  d < D,
 * so the image of one kv head is contiguous and a head-sharded receiver imports its own heads only.
 * `image` is a DEVICE pointer, 16-byte aligned: local memory, or a peer GPU's memory mapped into this
 * process (NVLink P2P), which makes export a direct remote write and import a direct remote read.
 * Both calls enqueue one gather / scatter kernel on `stream` and never synchronise.  The bits of K', V
 * are copied unchanged; positions are implicit (token t of the image is session token tok_begin + t on
 * export and session_len + t on import), so a receiver must import a session's images in order. */
SA_API int32_t sa_kv_wire_bytes(const sa_kv_pool *pool, int64_t n_tokens, size_t *out_bytes);
/* Tokens [tok_begin, tok_begin + n_tokens) of session `sid` -> image.  The session is not changed.
 * SA_ERR_INVALID_ARG if the range is not inside the session, SA_ERR_WORKSPACE_TOO_SMALL if
 * image_bytes < sa_kv_wire_bytes(n_tokens). */
SA_API int32_t sa_kv_session_export(sa_kv_pool *pool, int32_t sid, int64_t tok_begin, int64_t n_tokens, void *image,
                             size_t image_bytes, void *stream);
/* Appends n_tokens tokens to session `sid` from an image that holds `src_heads` kv heads, taking heads
 * [head_begin, head_begin + pool's Hkv).  Page allocation, copy-on-write of a shared partial page and
 * failure behaviour are sa_rope_kv_append's (SA_ERR_OUT_OF_PAGES changes nothing); nothing is rotated. */
SA_API int32_t sa_kv_session_import(sa_kv_pool *pool, int32_t sid, int64_t n_tokens, const void *image, int32_t src_heads,
                             int32_t head_begin, void *stream);

/* The same two operations for MANY sessions in one call and one kernel launch each (a PD hand-over moves every request of a
 * batch; one launch per session leaves the copy host- and launch-bound).  Range i is tokens [tok_begin[i], tok_begin[i] +
 * n_tokens[i]) of session sids[i] and has its own image (images[i], image_bytes[i]; any mix of local and peer addresses);
 * a session may appear in several ranges of an export.  Import: session sids[i] (each at most once) grows by n_tokens[i]
 * tokens from images[i]; page allocation is all-or-nothing over the whole call.  sids, tok_begin, n_tokens, images,
 * image_bytes are HOST arrays of n entries, copied before the call returns; at most 4 x max_sessions ranges per export (a list
 * longer than one metadata slab of the pool holds -- about 2 x max_sessions + num_pages / 8 + 2000 ranges -- is enqueued as several
 * launches; the images do not depend on that). */
SA_API int32_t sa_kv_sessions_export(sa_kv_pool *pool, int32_t n_ranges, const int32_t *sids, const int64_t *tok_begin,
                              const int64_t *n_tokens, void *const *images, const size_t *image_bytes, void *stream);
SA_API int32_t sa_kv_sessions_import(sa_kv_pool *pool, int32_t n_sessions, const int32_t *sids, const int64_t *n_tokens,
                              const void *const *images, int32_t src_heads, int32_t head_begin, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* SMOOTHAGENT_H_ */
