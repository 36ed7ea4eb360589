/*
 * spork.h -- C ABI of libspork: the data-parallel hot path behind Spork's
 * prefix-cache fork (arxiv/paper_2607_03333), B200 / sm_100a.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md at build time):
 *   - a probe is FORKED from the main stream so that its prompt prefix is a KV
 *     cache hit ("Fork a completions request ... {D1 cache hit}", Algorithm 1
 *     step 6; section 4.1);
 *   - main and probe(s) DECODE concurrently over the shared prefix
 *     (Fig. 7 text);
 *   - D3 VERIFIES the k probe tokens as drafts "in the same decode step" and
 *     accepts the longest greedy-matching prefix (section 4.3);
 *   - a probe that ends / is rejected / times out / is superseded is RELEASED
 *     (PAPER.md:211, :503, :585).
 * The paper gives no mechanism below those events; the paged-KV design here
 * (block tables, page refcounts, cascade split, LSE merge) follows
 * BASELINE.json `north_star` and the readings A-1..A-25 in DESIGN.md.
 *
 * Conventions
 *   - Every function returns 0 (SPORK_OK) or a negative spork error code.
 *     Nothing throws or aborts across this boundary.
 *   - "host" pointers are read (or written) before the call returns; the caller
 *     may reuse them immediately.  "device" pointers are CUDA device memory,
 *     caller-owned, used in stream order on `stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).
 *   - All state-changing calls and attention calls on one handle must be issued
 *     from one thread and onto one stream (or onto streams the caller orders).
 *     A handle is not thread-safe.
 *   - Batched state calls are all-or-nothing: on any error no state changes.
 *   - The library never synchronises the stream on the success path, with one
 *     documented exception: when its lower bound on free pages cannot prove
 *     that an allocating call fits, it reads the exact device-side free count
 *     (one 4-byte copy).  (Which pages the members of a fork group share is
 *     known on the host from the fork lineage; nothing is read back for it.)
 *   - Page size is 16 tokens.  Page allocation is deterministic: the lowest
 *     free page id first, requests in array order, positions ascending
 *     (reading A-1), so block tables and refcounts are unique.
 */
#ifndef SPORK_H
#define SPORK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPORK_PAGE_SIZE 16

#define SPORK_OK 0
#define SPORK_ERR_INVALID (-1)      /* bad argument / shape / unsupported config  */
#define SPORK_ERR_OOM (-2)          /* not enough free pages (nothing changed)     */
#define SPORK_ERR_NO_SLOT (-3)      /* not enough free sequence slots              */
#define SPORK_ERR_TOO_LONG (-4)     /* sequence would exceed max_pages_per_seq     */
#define SPORK_ERR_INVALID_SEQ (-5)  /* id out of range, not live, or repeated      */
#define SPORK_ERR_SHARED (-6)       /* truncate would expose a shared partial page */
#define SPORK_ERR_CUDA (-7)         /* a CUDA runtime call failed                  */
#define SPORK_ERR_DEVICE (-8)       /* device-side consistency check tripped       */
#define SPORK_ERR_STALE (-9)        /* a captured turn ran: call spork_turn_sync    */
#define SPORK_ERR_LIMIT (-10)       /* size beyond a no-allocation entry point's fixed maximum */

#define SPORK_F32 0
#define SPORK_BF16 1
#define SPORK_E4M3 2   /* FP8-KV variant (reading B-4): K and V are e4m3
                          bytes ("fn": bias 7, subnormals, no infinities, s.1111.111 = NaN); Q is BF16 */

typedef struct spork_ctx spork_ctx;

typedef struct spork_config {
    int32_t dtype;             /* SPORK_F32 | SPORK_BF16: storage type of K, V and Q;
                                  SPORK_E4M3: K and V are e4m3 bytes, Q is bf16            */
    int32_t num_q_heads;       /* Hq                                                    */
    int32_t num_kv_heads;      /* Hkv, divides Hq; q head h reads kv head h/(Hq/Hkv)    */
    int32_t head_dim;          /* D: multiple of 32, <= 256                             */
    int32_t page_size;         /* must be SPORK_PAGE_SIZE                               */
    int32_t num_pages;         /* NP: pages in each pool                                */
    int32_t max_seqs;          /* sequence slots                                        */
    int32_t max_pages_per_seq; /* block-table row length                                */
    float scale;               /* softmax scale (1/sqrt(D)); scores = scale * <q,k>     */
} spork_config;

/* Bytes of one page in ONE pool (K or V): Hkv * 16 * D * sizeof(K/V element). */
size_t spork_page_bytes(const spork_config *cfg);

/*
 * create / destroy.
 * k_pool, v_pool: device, caller-owned (allocated with e.g. PyTorch), each
 * num_pages * spork_page_bytes() bytes, 256-byte aligned, contents arbitrary.
 * Logical layout of a pool is [num_pages][Hkv][16][D]; the arrangement of the
 * 16 x D elements inside one (page, kv head) block is library-defined (for
 * bf16 with D % 64 == 0, and for e4m3 with D % 128 == 0, it is a 128-byte-swizzled
 * shared-memory image, so a block is staged with one bulk copy).  Write
 * pools only through spork_append / spork_fork; read them through
 * spork_read_kv.  The library owns block tables, refcounts and workspace.
 * Errors: SPORK_ERR_INVALID (shapes), SPORK_ERR_CUDA.
 */
int spork_create(const spork_config *cfg, void *k_pool, void *v_pool, spork_ctx **out);
int spork_destroy(spork_ctx *ctx);

/* n new empty sequences in the lowest free slots; ids_out: host int32[n]. */
int spork_seq_create(spork_ctx *ctx, int n, int32_t *ids_out);

/*
 * append: the "prefill / decode wrote KV" event (Algorithm 1 steps 1-5,
 * PAPER.md:257-261); also how draft KV is placed before verify.
 * seq_ids, n_tokens: host int32[n] (a sequence may repeat; requests apply in
 * array order).  k_src, v_src: device, [sum n_tokens][Hkv][D] in cfg.dtype.
 * A page is allocated whenever a sequence crosses a page boundary.
 * Errors: INVALID_SEQ, TOO_LONG, OOM.
 */
int spork_append(spork_ctx *ctx, int n, const int32_t *seq_ids, const int32_t *n_tokens,
                 const void *k_src, const void *v_src, void *stream);

/*
 * fork: Algorithm 1 step 6.  Child i clones parent_ids[i]'s
 * block table: the floor(len/16) full pages are shared (refcount + 1 each),
 * a partially filled tail page is duplicated into a fresh page (whole page,
 * K and V), child length = parent length.  Parents must be live before the
 * call; a parent may repeat.  Children take the lowest free slots in request
 * order; child_ids_out: host int32[n].  The parent is unchanged.
 * Errors: INVALID_SEQ, NO_SLOT, OOM.
 */
int spork_fork(spork_ctx *ctx, int n, const int32_t *parent_ids, int32_t *child_ids_out,
               void *stream);

/*
 * release: the probe finished / was rejected / timed out / was superseded
 * or the main stream finished.  Every block-table
 * entry drops one reference; pages reaching 0 are free.  A parent may be
 * released before its children.  Errors: INVALID_SEQ (not live, or repeated
 * within the batch).
 */
int spork_release(spork_ctx *ctx, int n, const int32_t *seq_ids, void *stream);

/*
 * truncate: rollback of rejected drafts (section 4.3 step 3).
 * new_len: host int32[n], 0 <= new_len <= len.  Frees whole pages beyond
 * ceil(new_len/16).  Errors: INVALID_SEQ, INVALID, SHARED (the kept tail page
 * is partially filled and has refcount > 1).
 */
int spork_truncate(spork_ctx *ctx, int n, const int32_t *seq_ids, const int32_t *new_len,
                   void *stream);

/*
 * decode attention, q_len = 1 (main and probes decode in one
 * batch).  The batch is seq_ids[group_indptr[n_groups]] (host int32), split
 * into fork groups by group_indptr (host int32[n_groups+1]); a group of 1 is
 * plain paged decode.  For each group the library finds the leading pages
 * its members have in common -- all of them, and, level by level, every
 * subset that shares more (probes forked at successive positions) -- and
 * reads each shared run from HBM once for the members that share it
 * (cascade); the result does not depend on the grouping beyond rounding.  q: device [n_seq][Hq][D] cfg.dtype.  out: device fp32
 * [n_seq][Hq][D].  lse: device fp32 [n_seq][Hq], natural log of
 * sum_t exp(scale * <q, k_t>).  Row i attends all len(seq_ids[i]) tokens; an
 * empty sequence yields out = 0, lse = -inf.
 * Errors: INVALID, INVALID_SEQ.
 */
int spork_decode_attn(spork_ctx *ctx, int n_groups, const int32_t *group_indptr,
                      const int32_t *seq_ids, const void *q, float *out, float *lse,
                      void *stream);

/*
 * verify attention (section 4.3 step 2): sequence i has
 * k_i = q_indptr[i+1] - q_indptr[i] draft positions whose KV are already its
 * last k_i tokens; query row j of sequence i attends tokens
 * t <= len_i - k_i + j.  q: device [sum k][Hq][D]; out fp32 [sum k][Hq][D];
 * lse fp32 [sum k][Hq].  Errors: INVALID (k_i < 1 or k_i > len_i), INVALID_SEQ.
 */
int spork_verify_attn(spork_ctx *ctx, int n_groups, const int32_t *group_indptr,
                      const int32_t *seq_ids, const int32_t *q_indptr, const void *q,
                      float *out, float *lse, void *stream);

/*
 * Host-buffer forms (what bench.py's `e2e` times): q_host, out_host, lse_host
 * are HOST buffers (pinned for full speed); the copies run on `stream` inside
 * the call, and the call returns after the results have landed.
 */
int spork_decode_attn_host(spork_ctx *ctx, int n_groups, const int32_t *group_indptr,
                           const int32_t *seq_ids, const void *q_host, float *out_host,
                           float *lse_host, void *stream);
int spork_verify_attn_host(spork_ctx *ctx, int n_groups, const int32_t *group_indptr,
                           const int32_t *seq_ids, const int32_t *q_indptr, const void *q_host,
                           float *out_host, float *lse_host, void *stream);

/* ---- synchronous export (parity checks; each call synchronises) ----------- */
/* len_out: host int32 (-1 if the slot is not live); table_out: host
 * int32[ceil(len/16)] read from the DEVICE block table. */
int spork_export(spork_ctx *ctx, int32_t seq, int32_t *len_out, int32_t *table_out);
/* host_out: host int32[num_pages], the device refcounts. */
int spork_export_refcounts(spork_ctx *ctx, int32_t *host_out);
/* logical K/V of tokens [t0, t0+n) of one sequence; k_out, v_out: HOST
 * [n][Hkv][D] cfg.dtype. */
int spork_read_kv(spork_ctx *ctx, int32_t seq, int32_t t0, int32_t n, void *k_out, void *v_out);
/* device-side free page count (synchronises). */
int spork_free_pages(spork_ctx *ctx, int32_t *out);
/* synchronises and returns the sticky device error word (SPORK_OK if none). */
int spork_status(spork_ctx *ctx);

/* ---- introspection (bench / tests) --------------------------------------- */
typedef struct spork_plan_info {
    int32_t n_items;        /* work items of the last attention call                */
    int32_t n_prefix_items; /* of which shared-prefix items                         */
    int32_t chunk_tokens;   /* split-KV chunk length                                */
    int32_t grid;           /* CTAs launched by the attention kernel                */
    int32_t kernel;         /* 0 = simt (fp32 / generic); bf16, D = 128: 1 = mma.sync,
                               2 = tcgen05, 3 = both (many-row items on tcgen05)     */
    int32_t plan_cached;    /* 1 if the last call reused the previous plan          */
    int64_t unique_tokens;  /* sum_groups (shared + sum_members private) tokens     */
    int64_t naive_tokens;   /* sum_members len                                      */
    int64_t partial_rows;   /* rows of split-KV workspace written                   */
    int32_t launches;       /* kernels launched by the last attention call          */
    int32_t n_umma_items;   /* of n_items, those run by the tcgen05 kernels         */
    int32_t n_two_pipe_items; /* of those, items on the second tcgen05 list (knob)   */
    int32_t stream_k;       /* 1: equal-work contiguous schedule    */
    float plan_host_us;     /* host time of the last plan BUILD (a cache miss), us   */
    int32_t plan_builds;    /* plans built on this handle so far (cache misses)      */
    int32_t n_levels;       /* deepest cascade level of the last plan (1 = single)   */
    int32_t reserved;
} spork_plan_info;
int spork_last_plan(spork_ctx *ctx, spork_plan_info *out);
/* kernels launched by the last state call (append / fork / release / truncate) */
int spork_last_launches(spork_ctx *ctx);

/*
 * Kernel timing for bench.py's roofline: when enabled, the attention calls
 * record CUDA events on `stream` around the attention kernel and around the
 * merge kernel, and spork_fork records them around fork_clone_kernel (its
 * dominant kernel; merge_ms is then 0).  spork_last_kernel_ms synchronises on
 * them and returns the two durations of the last such call (milliseconds).
 * Off by default (no events).
 */
int spork_set_timing(spork_ctx *ctx, int enable);
int spork_last_kernel_ms(spork_ctx *ctx, float *attn_ms, float *merge_ms);

/*
 * Partial-token accept + rollback (section 4.3: "the first k matching tokens are
 * accepted").  Sequence seq_ids[i] holds k_i = q_indptr[i+1] - q_indptr[i]
 * draft tokens as its LAST k_i tokens (appended before spork_verify_attn).  draft_tokens and
 * target_tokens are DEVICE int32 arrays of sum k_i entries, ragged by q_indptr: the drafts, and the
 * target model's greedy token at each draft position (computed by the caller's LM head from the
 * verify output; not part of this library).  For every sequence: accept_len_i = number of leading
 * positions with draft == target (one warp per sequence); the rejected drafts' KV is rolled back as
 * spork_truncate(seq_i, len_i - (k_i - accept_len_i)) does (whole pages beyond the new length are
 * freed).  accept_len_out: HOST int32[n], written before return.  seq_ids, q_indptr: host, read
 * before return.  Synchronises `stream` once (the host mirrors lengths).  Errors: SPORK_ERR_INVALID
 * (k_i < 1, k_i > len_i, null pointers), SPORK_ERR_INVALID_SEQ, SPORK_ERR_SHARED as for
 * spork_truncate; on a validation error nothing changes.
 */
int spork_accept(spork_ctx *ctx, int n, const int32_t *seq_ids, const int32_t *q_indptr,
                 const int32_t *draft_tokens, const int32_t *target_tokens, int32_t *accept_len_out,
                 void *stream);

/*
 * D2 confidence score (Eq. 2): for each of n_spans tool-name
 * spans, c = min_{i=2..L} exp(l_i), l_i the log-probability of the TOP-1 token at position i, i.e.
 * min_i 1 / sum_v exp(x_iv - max_v x_iv).  logits: DEVICE fp32 [n_pos][vocab], row-major, rows of span
 * s are [span_indptr[s], span_indptr[s+1]) (span_indptr: HOST int32[n_spans + 1], starts at 0, read
 * before return); the first row of a span is skipped (i starts at 2), a span of <= 1 rows gives 1.
 * confidence_out: DEVICE fp32[n_spans].  Stream-ordered, no synchronisation.  The gate itself
 * (c >= theta) is the caller's.  Errors: SPORK_ERR_INVALID (null pointers, vocab < 1,
 * decreasing span_indptr).
 */
int spork_confidence(spork_ctx *ctx, int n_spans, const int32_t *span_indptr, const float *logits,
                     int vocab, float *confidence_out, void *stream);

/*
 * The same score (Eq. 2) for callers that cannot allocate: code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc.  The call makes two kernel launches
 * on `stream` and nothing else -- no cudaMalloc / cudaFree or allocating library routine, no staging
 * copy, no synchronisation, no host read of device memory -- and needs no context.  The per-(row,
 * vocabulary slice) partial sums that spork_confidence keeps in a buffer it grows live here in ONE
 * file-scope device array of 2 * SPORK_CONFIDENCE_STATIC_MAX_ROWS float2 (256 KiB), which every GPU
 * that loads libspork holds until the process exits.
 *   span_indptr    DEVICE int32[n_spans + 1] (spork_confidence reads it on the host): non-decreasing,
 *                  span_indptr[0] = 0, span_indptr[n_spans] = n_pos.  Not checked (it is device memory);
 *                  values outside this contract give undefined scores (the kernels clamp them to the
 *                  rows that exist: nothing outside the array or the logits is read).
 *   n_pos          rows of logits; at most SPORK_CONFIDENCE_STATIC_MAX_ROWS, else SPORK_ERR_LIMIT and
 *                  nothing is launched.
 *   logits         DEVICE fp32 [n_pos][vocab], row-major; confidence_out: DEVICE fp32[n_spans].
 * Results equal spork_confidence's up to the rounding of a different slicing of the vocabulary.
 * The array is shared by every call on the device and keeps the last call's contents: each slot a call
 * reads it has written itself (nothing needs to start at zero), but two calls that OVERLAP on the GPU
 * (different streams, parallel graph branches) race on it -- order them.  The first call on a device
 * resolves the array's device address (cudaGetSymbolAddress, with that device current) and must be
 * made outside stream capture; n_spans = 0 does only that.  The current device must be the one
 * `stream`, the pointers and later calls belong to.  Errors: SPORK_ERR_INVALID (null pointers,
 * negative sizes, vocab < 1), SPORK_ERR_LIMIT (n_pos beyond the maximum, device ordinal >= 64),
 * SPORK_ERR_CUDA.
 */
#define SPORK_CONFIDENCE_STATIC_MAX_ROWS 16384
int spork_confidence_static(int n_spans, const int32_t *span_indptr, int n_pos, const float *logits,
                            int vocab, float *confidence_out, void *stream);

/*
 * Tuning knob of the planner (bf16, D = 128 contexts only): a segment -- a fork group's shared
 * prefix or one sequence's private tail -- whose query rows x GQA heads per KV head number at
 * least `min_rows` is run by the tcgen05 (TMEM) kernel in row blocks of 128, the others by the
 * mma.sync kernel.  Default 1: everything runs on the tcgen05 kernel (measured at least as fast
 * as any split on every BASELINE.json config); a value above the largest row count sends
 * everything to the mma.sync kernel.  Results do not depend on it beyond rounding.  Invalidates the
 * cached plan.  SPORK_ERR_INVALID on a null context.
 */
int spork_set_tensor_path_min_rows(spork_ctx *ctx, int min_rows);
/*
 * Tuning knob: which tcgen05 kernel variant runs a tensor-path segment of more than 128 rows
 * (verify: drafts x group members x GQA heads).  mode 0 (default): the one-pipe kernel in row
 * blocks of 128, each block re-reading the K/V tiles through L2.  mode 1: row blocks of 256 on
 * the two-pipe variant (one CTA per SM, two softmax pipes share one stream of K/V tiles).
 * mode 2: row blocks of 128 on the split-row variant (each row's 64 scores of a tile shared by
 * two threads, 8 softmax warps per CTA).  Measured on BASELINE.json config 4: mode 0 is equal or
 * faster (k = 8: 342 / 410 / 430 us, k = 16: 671 / 730 / 712 us for modes 0 / 1 / 2), hence the
 * default; the variants stay for the next round's tuning and are covered by the parity tests.
 * Results do not depend on the mode beyond rounding.  Other values are read as 0.  Invalidates
 * the cached plan.
 */
int spork_set_many_row_variant(spork_ctx *ctx, int mode);
/*
 * Tuning knob: allow (default) or forbid the stream-K schedule.  Allowed: when every segment of
 * a call is a single row block of the tcgen05 kernel (every decode call on a bf16, D = 128
 * context; verify with few drafts), the (segment, kv head) streams are laid end to end and cut
 * into one contiguous, equal-cost run per persistent CTA.  Forbidden, or for other calls: equal
 * chunks per segment, longest-processing-time-first onto the CTAs.  Results do not depend on it
 * beyond rounding.  Invalidates the cached plan.
 */
int spork_set_stream_k(spork_ctx *ctx, int enable);

/*
 * Tuning knob: the deepest cascade the planner builds for a fork group (default 7).  A group is
 * planned as a trie: every set of members that holds further pages in common beyond what the
 * whole group shares (probes forked from the main stream at successive CoT positions, Algorithm 1
 * steps 4-6) gets a shared segment of its own, read from HBM once for that set.
 * max_levels = 1: only the group-wide prefix is shared, deeper sharing is read once per member.
 * Results do not depend on it beyond rounding.  Invalidates the cached plan.
 */
int spork_set_cascade_levels(spork_ctx *ctx, int max_levels);

/*
 * Multi-layer step (the Qwen3 models the paper serves have 36 / 64 / 48
 * layers).  Block tables, refcounts and lengths are per SEQUENCE, not per layer: one
 * handle serves every layer's K/V pools.
 *   spork_layers: registers the pools of layers 0 .. n_layers-1 (host arrays of device pointers, each
 *     pool sized and aligned like create's; k_pools[0] / v_pools[0] must be create's pools).  From
 *     then on spork_fork duplicates a partially filled tail page in EVERY layer.
 *   spork_append allocates pages and writes layer 0's K/V; spork_write_kv_layer writes the K/V of the
 *     LAST n_tokens[i] tokens of seq_ids[i] (already appended) into layer `layer`'s pools (k_src,
 *     v_src: device, [sum n_tokens][Hkv][D]).  Errors: INVALID (n_tokens[i] > len), INVALID_SEQ.
 *   spork_decode_attn_layers / spork_verify_attn_layers: ONE plan, then n_layers x (attention kernel,
 *     merge kernel) back to back, layer l on pools l with q[l] -> out[l], lse[l] (HOST arrays of
 *     n_layers device pointers, shapes as in the single-layer calls).  Each kernel is launched
 *     programmatically behind the previous one, so launch latency and prologues overlap.  All q[l]
 *     must be ready when the call is made.
 */
int spork_layers(spork_ctx *ctx, int n_layers, void *const *k_pools, void *const *v_pools, void *stream);
int spork_write_kv_layer(spork_ctx *ctx, int layer, int n, const int32_t *seq_ids, const int32_t *n_tokens,
                         const void *k_src, const void *v_src, void *stream);
int spork_decode_attn_layers(spork_ctx *ctx, int n_layers, int n_groups, const int32_t *group_indptr,
                             const int32_t *seq_ids, const void *const *q, float *const *out,
                             float *const *lse, void *stream);
int spork_verify_attn_layers(spork_ctx *ctx, int n_layers, int n_groups, const int32_t *group_indptr,
                             const int32_t *seq_ids, const int32_t *q_indptr, const void *const *q,
                             float *const *out, float *const *lse, void *stream);

/*
 * One partial-token-accept turn without a host round trip, for CUDA-graph capture (SURVEY.md 8(f) NEXT-1:
 * "end-to-end fork -> decode -> verify -> accept -> rollback step under one CUDA graph"; "in
 * the same decode step (no separate verification pass)"; the decode loop of Algorithm 1 steps 4-5,
 * PAPER.md:260-261).  The calls below enqueue ONLY kernel launches over buffers that do not move -- no
 * host copy, no synchronisation, every decision (pages taken in request order: reading A-1; accept
 * length; rollback) taken by kernels from the DEVICE lengths -- so the caller may capture any sequence
 * of them, together with its own kernels, with cudaStreamBeginCapture (or torch.cuda.graph) on `stream`
 * and replay the graph turn after turn:
 *     spork_turn_append(t, 0, ...)   k_i draft tokens to every sequence (k_src, v_src: device,
 *                                    [sum k_i][Hkv][D], ragged by q_indptr)
 *     spork_turn_verify(t, ...)      as spork_verify_attn over the turn's batch (q [sum k_i][Hq][D])
 *     spork_turn_accept(t, ...)      accept_len_i = leading positions with draft == target; the rejected
 *                                    drafts are rolled back as spork_accept does; accept_len_dev: DEVICE
 *                                    int32[n] or NULL
 *     spork_turn_append(t, 1, ...)   one token to every sequence (k_src, v_src: [n][Hkv][D])
 *     spork_turn_decode(t, ...)      as spork_decode_attn over the turn's batch (q [n][Hq][D])
 * spork_turn_prepare (not capturable) fixes the batch: groups, sequences (each once, non-empty) and the
 * number of drafts k_i = q_indptr[i+1] - q_indptr[i] in [1, 64] per sequence; it builds the two attention
 * plans and uploads the descriptors.  The plans stay valid while sequences only grow (a turn nets
 * accept_len + 1 tokens) and no other call changes the batch's sharing (fork / release / truncate of any
 * sequence: the turn's calls then return SPORK_ERR_INVALID; prepare again).
 * From the first turn call on the host's copy of the lengths is stale: every other state or attention
 * call returns SPORK_ERR_STALE until spork_turn_sync (which synchronises `stream`, reads the lengths and
 * the free-page count back, and returns SPORK_ERR_DEVICE if a turn ran out of pages or block-table row --
 * such an append leaves the state untouched, as the host path does -- or if spork_turn_accept was asked to
 * roll a sequence back below its length at spork_turn_prepare, i.e. to reject drafts the turn did not
 * append: that sequence is left alone).  After a sync the graph can go on
 * being replayed.  Errors: INVALID, INVALID_SEQ, STALE, CUDA.
 */
typedef struct spork_turn spork_turn;
int spork_turn_prepare(spork_ctx *ctx, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
                       const int32_t *q_indptr, void *stream, spork_turn **out);
int spork_turn_append(spork_turn *t, int which, const void *k_src, const void *v_src, void *stream);
int spork_turn_verify(spork_turn *t, const void *q, float *out, float *lse, void *stream);
int spork_turn_accept(spork_turn *t, const int32_t *draft_tokens, const int32_t *target_tokens,
                      int32_t *accept_len_dev, void *stream);
int spork_turn_decode(spork_turn *t, const void *q, float *out, float *lse, void *stream);
int spork_turn_sync(spork_turn *t, void *stream);
int spork_turn_destroy(spork_turn *t);

/*
 * Bench support: one read-only pass over `bytes` bytes at `buf` (device, 16-byte aligned; whole 16 KiB
 * chunks are read), streamed like the attention kernel streams K/V (bulk copies into shared memory from
 * 2 persistent CTAs per SM), launched on `stream`; the caller times it with events.  bench.py reports the rate it reaches (`read_peak`) beside
 * MEASURED_PEAKS.json's copy figure: the attention kernels are read streams (SURVEY.md 8(d) asks for GB/s
 * against the box's measured bandwidth).  Errors: SPORK_ERR_INVALID.
 */
int spork_hbm_read_probe(spork_ctx *ctx, const void *buf, size_t bytes, void *stream);

const char *spork_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* SPORK_H */
