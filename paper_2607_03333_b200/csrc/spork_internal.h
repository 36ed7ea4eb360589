// Internal declarations of libspork (CUDA path).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "spork.h"

namespace spork {

constexpr int PS = SPORK_PAGE_SIZE;  // tokens per page

// ---------------------------------------------------------------------------
// Work list (built on the host by plan.cu, consumed by the attention kernels)
// ---------------------------------------------------------------------------
// One item = one (segment, split, kv head, row block): `nrows` query rows
// against tokens [tok0, tok1) of the sequence in slot `table_seq`.
// Logical row r (rb0 <= r < rb0 + nrows) is q head (kvh * G + r % G) of the segment's (r / G)-th
// q row: q row qrow0 + r / G, or rowmap[rowmap + r / G] when the segment's rows are not
// consecutive in the call (a sub-tree of a fork group).  Token t is visible to row r iff
// t <= lim0 + r / G (lim0 = INT_MAX/2 for shared segments: no mask).
// Items of a private tail carry flags: ITEM_LEN_LIM: lim0 = len[table_seq] - lim_k, and on the
// tail's last piece ITEM_LEN_TOK1: tok1 = len[table_seq], both read from the DEVICE lengths when the
// kernel runs -- a plan stays valid while its sequences grow by appended tokens.
struct WorkItem {
    int32_t table_seq;
    int32_t tok0;       // multiple of 16
    int32_t tok1;       // exclusive
    int32_t kvh;
    int32_t qrow0;
    int32_t rb0;
    int32_t nrows;      // <= 64 (mma.sync / simt path), <= 128 / 256 (tcgen05 kernel, one / two pipes)
    int32_t lim0;
    int32_t part_base;  // partial row index of logical row rb0
    int32_t flags;      // ITEM_*
    int32_t lim_k;
    int32_t rowmap;     // -1: rows are consecutive from qrow0
};
static_assert(sizeof(WorkItem) == 48, "WorkItem layout");
enum : int32_t { ITEM_LEN_LIM = 1, ITEM_LEN_TOK1 = 2 };

// A stream = (segment, kv head): the partials of its rows.  Partial row index of
// (split s, row i of the stream) = part_base + s * stride + i, rows ordered (q row, GQA head).
// Different kv heads of one segment may be cut at different places (stream-K schedule).
struct StreamDesc {
    int32_t part_base, nsplit, stride, pad;
};
static_assert(sizeof(StreamDesc) == 16, "StreamDesc layout");

// Per q row: the segments it has partials in -- one per cascade level it shares with other members
// of its fork group, plus its private tail: refs [ref0, ref0 + nref).  A ref names the segment's
// stream of kv head 0 (kv head h is stream + h) and the row's offset (q index in the segment) * G.
struct RowRef {
    int32_t stream, off;
};
struct QRowDesc {
    int32_t ref0, nref;
};
static_assert(sizeof(QRowDesc) == 8 && sizeof(RowRef) == 8, "merge descriptor layout");
constexpr int MAX_ROW_REFS = 8;     // deepest cascade: 7 shared levels + the private tail

// One append request as the append kernels read it (built on the host by spork_append, on the device by
// the captured turn: turn.cu)
struct AppendDesc {
    int32_t seq, old_len, n_tok, tok_off;
    int32_t free_off;   // index into free_list of this request's first new page
    int32_t n_new;      // pages this request allocates
    int32_t final_len;  // >= 0: this request writes len[seq] (last request of the sequence)
    int32_t pad;
};

// Host lineage of a sequence: which incarnation allocated each of its pages, run-length encoded.
// Pages [r[i-1].end, r[i].end) were allocated by incarnation r[i].uid (a fresh uid is drawn at
// seq_create, at fork (for the child) and at truncate).  Two sequences hold the same physical page at
// index j exactly when their labels at j are equal, so the common leading pages of any set of
// sequences follow from the host alone (no device read-back).  More than MAX_RUNS runs: the deepest
// ones are folded into a private run, which can only under-state sharing.
struct Lineage {
    static constexpr int MAX_RUNS = 8;
    int32_t n = 0;
    int32_t end[MAX_RUNS];
    uint64_t uid[MAX_RUNS];
    int pages() const { return n ? end[n - 1] : 0; }
};

// ---------------------------------------------------------------------------
// staging ring: pinned host + device scratch for per-call descriptors
// ---------------------------------------------------------------------------
struct StageSlot {
    void *h = nullptr;
    void *d = nullptr;
    size_t cap = 0;
    cudaEvent_t ev = nullptr;
    bool pending = false;
};

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
};

struct Plan {
    bool valid = false;
    // cache keys
    uint64_t structure_epoch = 0, len_epoch = 0;
    bool verify = false;
    std::vector<int32_t> group_indptr, seq_ids, q_indptr;
    std::vector<int32_t> base_len;   // lengths the plan was built for; it stays valid while
                                     // base_len <= len < base_len + GROW_WINDOW for every sequence
    bool growable = false;
    int64_t base_unique = 0, base_naive = 0;
    // device copy: ONE buffer
    //   items   = [n_items of the mma.sync / simt path][n_items_umma of the tcgen05 kernel, <= 128 rows]
    //             [n_items_umma2 of the two-pipe tcgen05 kernel, <= 256 rows]
    //   cta_ptr = int32[grid + 1], int32[grid_umma + 1], int32[grid_umma2 + 1]: CTA b of a kernel
    //             runs items [cta_ptr[b], cta_ptr[b + 1]) of its own list
    DevBuf blob;
    const WorkItem *d_items = nullptr;
    const QRowDesc *d_qdesc = nullptr;
    const RowRef *d_refs = nullptr;
    const StreamDesc *d_streams = nullptr;
    const int32_t *d_cta_ptr = nullptr;
    const int32_t *d_rowmap = nullptr;
    int n_items = 0, n_qrows = 0, grid = 0;
    int n_items_umma = 0, grid_umma = 0;
    int n_items_umma2 = 0, grid_umma2 = 0;
    int variant2 = 1;           // kernel of the second tcgen05 list: 1 two pipes, 2 split rows
    spork_plan_info info{};
};

}  // namespace spork

struct spork_ctx {
    spork_config cfg;
    int G;               // Hq / Hkv
    int elt;             // bytes per K / V element
    int q_elt;           // bytes per Q element (= elt, except e4m3 KV: bf16 queries)
    int swizzled;        // D * elt % 128 == 0 (bf16, e4m3): 128B-swizzled page-head blocks
    size_t head_block;   // bytes of one (page, kv head) block in one pool
    size_t page_bytes;   // bytes of one page in one pool
    int table_stride;    // int32 per block-table row (max_pages_per_seq rounded up to 4)
    int num_sms;
    void *k_pool, *v_pool;

    // device state
    int32_t *d_refcount;  // [num_pages]
    int32_t *d_table;     // [max_seqs][table_stride]
    int32_t *d_len;       // [max_seqs]
    int32_t *d_counters;  // [0] free pages, [1] sticky error, [2..] scratch
    int32_t *d_free_list; // [free_list_cap] lowest free ids, ascending
    int32_t *d_scan;      // block counts for the free-page scan
    size_t free_list_cap;

    // host mirrors (lengths and slot occupancy only; never refcounts or tables)
    std::vector<int32_t> h_len;
    std::vector<uint8_t> h_live;
    std::vector<int32_t> h_shared_upto;  // pages below this index MAY be shared
    std::vector<uint64_t> h_fork_key;    // (fork call, parent slot) the sequence was cloned by; 0: none / rolled back
    std::vector<int32_t> h_fork_nf;      // full pages it shared with its parent at that fork
    uint64_t fork_calls = 0;
    std::vector<int32_t> h_scratch;      // per-slot scratch (fork counts, evolving lens)
    std::vector<spork::Lineage> h_lin;   // page lineage per slot (see Lineage)
    std::vector<uint64_t> h_uid;         // current incarnation of the slot
    uint64_t next_uid = 1;
    int64_t free_lb;                     // lower bound on free pages
    bool mirror_stale = false;           // a captured turn ran: lengths live on the device only until spork_turn_sync
    bool fl_valid = false;               // d_free_list[fl_pos, fl_n) are still the lowest free ids (see take_free)
    int fl_pos = 0, fl_n = 0;
    int n_live;

    uint64_t structure_epoch, len_epoch;

    spork::StageSlot stage[8];
    int stage_next;

    spork::Plan plan;
    spork::DevBuf ws_o, ws_lse;   // split-KV partials
    spork::DevBuf io_q, io_out, io_lse;  // device buffers of the *_host calls
    spork::DevBuf ws_conf;               // per-(row, slice) partials of spork_confidence
    spork::DevBuf conf_desc;             // its device descriptors, cached while the spans stay the same
    std::vector<int32_t> conf_key;
    void *h_io = nullptr;         // pinned bounce (unused if caller memory is pinned)
    int last_launches;
    int plan_builds = 0;
    uint32_t smem_attr_done = 0;          // bit per kernel: cudaFuncSetAttribute(MaxDynamicSharedMemorySize) done on this device
    int timing = 0;
    int stream_k = 1;             // equal-work contiguous schedule when every segment is one row block
    int many_row_variant = 0;             // segments of > 128 rows: 0 default kernel, 1 two-pipe, 2 split-row kernel
    int umma_min_rows = 1;        // segments with at least this many rows take the tcgen05 path
    int cascade_levels = spork::MAX_ROW_REFS - 1;   // deepest cascade the planner builds (1: the group-wide prefix only)
    std::vector<void *> layer_k, layer_v;   // pools of layers 1.. (layer 0 = k_pool / v_pool), see spork_layers
    spork::DevBuf d_layer_pools;            // the same pointers on the device: k of layers 1.., then v of layers 1..
    cudaEvent_t t_ev[3] = {nullptr, nullptr, nullptr};
    bool t_valid = false;
};

namespace spork {

#define SPORK_CUDA(call)                                   \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return SPORK_ERR_CUDA;     \
    } while (0)

__host__ __device__ inline int ceil_div(int a, int b) { return (a + b - 1) / b; }
__host__ __device__ inline int pages_of(int len) { return (len + PS - 1) / PS; }

// staging.cu / api.cu
int stage_acquire(spork_ctx *c, size_t bytes, StageSlot **out);           // waits for the slot
int stage_commit(spork_ctx *c, StageSlot *s, size_t bytes, cudaStream_t st);  // H2D copy
int stage_done(spork_ctx *c, StageSlot *s, cudaStream_t st);              // record reuse event
int devbuf_reserve(DevBuf *b, size_t bytes, cudaStream_t st);

// alloc.cu
int launch_free_scan(spork_ctx *c, int need, cudaStream_t st);  // fills d_free_list[0..need)
int ensure_pages(spork_ctx *c, int64_t need, cudaStream_t st);  // OOM check (may sync)
int take_free(spork_ctx *c, int need, cudaStream_t st, int *off);  // ids at d_free_list[*off, *off + need)
int launch_append_small(spork_ctx *c, const AppendDesc *d_descs, int n, int need, const void *k_src,
                        const void *v_src, cudaStream_t st);


// plan.cu
int build_plan(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
               const int32_t *q_indptr, cudaStream_t st);

// lineage (alloc.cu keeps it up to date, plan.cu reads it)
void lineage_reset(spork_ctx *c, int s);                       // seq_create / release
void lineage_grow(spork_ctx *c, int s, int n_pages);           // append: pages [old, n_pages) are the slot's own
void lineage_fork(spork_ctx *c, int child, int parent, int len);
void lineage_truncate(spork_ctx *c, int s, int keep_pages);
int lineage_lcp(const Lineage &a, const Lineage &b);           // common leading pages
uint64_t lineage_label(const Lineage &a, int page);            // 0: no such page

// attention launchers: one layer = (K pool, V pool, q, out, lse)
struct LayerIO {
    const void *k_pool, *v_pool, *q;
    float *out, *lse;
};
int launch_attn_simt(spork_ctx *c, const LayerIO &io, cudaStream_t st);
// attn_api.cu: attention + merge kernels of the plan that is in c->plan, one layer
int launch_planned(spork_ctx *c, const LayerIO &io, cudaStream_t st);
int launch_merge(spork_ctx *c, const LayerIO &io, cudaStream_t st);
int attn_mma_grid(spork_ctx *c);
int launch_attn_umma(spork_ctx *c, const LayerIO &io, int np, bool programmatic, bool wait_prev, cudaStream_t st);
int attn_umma_grid(spork_ctx *c, int variant);
int launch_attn_mma(spork_ctx *c, const LayerIO &io, bool programmatic, cudaStream_t st);

// Swizzled (page, kv head) block, bf16 with D % 64 == 0: the block is a run of 1 KiB
// atoms of 8 token rows x 128 bytes (64 dims), ordered [row group r/8][dim half d/64];
// inside an atom the 16-byte chunk index is XORed with (row & 7).  This is at once the
// conflict-free ldmatrix image and the canonical 128B-swizzle operand layout of
// tcgen05.mma (K: K-major, V: MN-major; 8-row groups 2 * nhalf KiB apart), so one
// bulk copy per block stages it for either tensor path.
// byte offset of 16-byte chunk c (0 .. D/8) of token row r
__host__ __device__ inline int swz_chunk_off(int nhalf, int r, int c) {
    return (((r >> 3) * nhalf + (c >> 3)) << 10) + ((r & 7) << 7) + (((c & 7) ^ (r & 7)) << 4);
}
// element offset (in elements of `elt` bytes: 2 or 1 when swizzled) of (slot r, dim d) inside one
// (page, kv head) block
__host__ __device__ inline int head_block_off(int swizzled, int D, int elt, int r, int d) {
    if (!swizzled) return r * D + d;
    const int per_chunk = 16 / elt;
    return swz_chunk_off(D * elt >> 7, r, d / per_chunk) / elt + d % per_chunk;
}

#ifdef __CUDACC__
// The item as the kernel runs it: lengths that the plan left open are read from the device now.
__device__ __forceinline__ WorkItem load_item(const WorkItem *__restrict__ items, int idx,
                                              const int32_t *__restrict__ len) {
    WorkItem it = items[idx];
    if (it.flags) {
        const int L = len[it.table_seq];
        if (it.flags & ITEM_LEN_TOK1) it.tok1 = L;
        if (it.flags & ITEM_LEN_LIM) it.lim0 = L - it.lim_k;
    }
    return it;
}
// q row of logical row lr of the item
__device__ __forceinline__ int item_qrow(const WorkItem &it, const int32_t *__restrict__ rowmap, int lr, int G) {
    return it.rowmap < 0 ? it.qrow0 + lr / G : rowmap[it.rowmap + lr / G];
}
#endif

}  // namespace spork
