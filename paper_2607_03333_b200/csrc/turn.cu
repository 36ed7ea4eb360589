// libspork: one partial-token-accept turn with no host round trip, so that the caller can capture it
// in a CUDA graph and replay it ("in the same decode step (no
// separate verification pass)"; the loop of Algorithm 1 steps 4-5):
//
//     append k_i drafts  ->  verify attention  ->  [caller: LM head -> target tokens]  ->
//     accept (longest matching prefix) + rollback  ->  append 1 token  ->  decode attention
//
// spork_append / spork_accept decide on the HOST (which pages a request takes, how far a sequence is
// rolled back); here the same decisions are taken by kernels from the DEVICE lengths, so a turn is a
// fixed sequence of launches over buffers that do not move:
//   turn_append_plan_kernel   per request, from len[]: pages needed, exclusive scan in request order ->
//                             the AppendDesc array the ordinary append kernel reads (the lowest free ids in
//                             request order: reading A-1, same tables as the host path)
//   turn_accept_kernel        one warp per sequence: accept length, new length, drops the freed pages
//   the attention kernels     run two plans built once at spork_turn_prepare; their open-ended items
//                             follow the device lengths (spork_internal.h ITEM_LEN_*)
// The host mirror of the lengths is stale from the first turn call until spork_turn_sync.
#include <string.h>

#include <algorithm>
#include <new>
#include <utility>

#include "spork_internal.h"

using namespace spork;

struct spork_turn {
    spork_ctx *c = nullptr;
    int n_seq = 0, n_groups = 0;
    std::vector<int32_t> seq_ids, k, base_len, group_indptr, q_indptr;
    uint64_t structure_epoch = 0;
    Plan plan_v, plan_d;            // verify (k_i rows per sequence) and decode (one row) plans
    int need_ub[2] = {0, 0};        // upper bound on the pages an append of kind 0 (drafts) / 1 (one token) takes
    int total_tok[2] = {0, 0};
    // one device buffer: seq_ids[n], n_tok[2][n], tok_off[2][n], base_len[n], q_indptr[n + 1], AppendDesc[n]
    DevBuf dev;
    const int32_t *d_seq = nullptr, *d_ntok[2] = {nullptr, nullptr}, *d_tokoff[2] = {nullptr, nullptr};
    const int32_t *d_qi = nullptr, *d_base = nullptr;
    AppendDesc *d_descs = nullptr;
};

namespace {

// One block.  Request i appends n_tok[i] tokens to sequence seq[i] (each sequence once): pages it needs
// from its DEVICE length, exclusive scan over the requests (array order = allocation order, A-1).  If the
// free pages do not suffice or a sequence would outgrow its block-table row, nothing is appended
// (all-or-nothing, as on the host path) and the sticky error word is set.
__global__ void __launch_bounds__(256) turn_append_plan_kernel(const int32_t *__restrict__ seq,
                                                               const int32_t *__restrict__ n_tok,
                                                               const int32_t *__restrict__ tok_off, int n,
                                                               const int32_t *__restrict__ len, int max_pages,
                                                               int32_t *counters, AppendDesc *__restrict__ descs) {
    __shared__ int s_warp[8], s_carry, s_bad;
    if (threadIdx.x == 0) { s_carry = 0; s_bad = 0; }
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int b = 0; b < n; b += blockDim.x) {
        const int i = b + threadIdx.x;
        int need = 0, L = 0;
        if (i < n) {
            L = len[seq[i]];
            need = pages_of(L + n_tok[i]) - pages_of(L);
            if (pages_of(L + n_tok[i]) > max_pages) atomicExch(&s_bad, 1);
        }
        int x = need;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) s_warp[w] = x;
        __syncthreads();
        int base = s_carry;
        for (int j = 0; j < w; ++j) base += s_warp[j];
        if (i < n) descs[i] = AppendDesc{seq[i], L, n_tok[i], tok_off[i], base + x - need, need, L + n_tok[i], 0};
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) s_carry = base + x;
        __syncthreads();
    }
    const int total = s_carry;
    const bool fail = s_bad || total > counters[0];
    __syncthreads();
    if (fail) {
        for (int i = threadIdx.x; i < n; i += blockDim.x) {
            descs[i].n_tok = 0;
            descs[i].n_new = 0;
            descs[i].final_len = -1;
        }
        if (threadIdx.x == 0) atomicExch(&counters[1], 3);
    } else if (threadIdx.x == 0) {
        counters[0] -= total;
    }
}

// One warp per sequence: accept length = leading positions with draft == target, the
// rejected drafts' pages are dropped and the length is rolled back, all from the device length.  The kept
// tail page cannot be shared, and the new length cannot fall below the length at spork_turn_prepare, when
// the drafts are the tokens the turn appended; should either happen, the sequence is left alone and the
// sticky error word is set.
__global__ void __launch_bounds__(128) turn_accept_kernel(const int32_t *__restrict__ seq,
                                                          const int32_t *__restrict__ q_indptr,
                                                          const int32_t *__restrict__ draft,
                                                          const int32_t *__restrict__ target,
                                                          const int32_t *__restrict__ base_len, int n, int32_t *len,
                                                          int32_t *table, int table_stride, int32_t *refcount,
                                                          int32_t *counters, int32_t *__restrict__ accept_out) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n) return;
    const int b = q_indptr[w], e = q_indptr[w + 1], k = e - b;
    int a = k;
    for (int j0 = b; j0 < e; j0 += 32) {
        const int j = j0 + lane;
        const unsigned m = __ballot_sync(0xffffffffu, j < e && draft[j] != target[j]);
        if (m) {
            a = j0 - b + __ffs(m) - 1;
            break;
        }
    }
    if (accept_out && lane == 0) accept_out[w] = a;
    const int s = seq[w], L = len[s], newL = L - (k - a);
    if (newL == L) return;
    int32_t *row = table + (size_t)s * table_stride;
    // (below the length the plans were built for, their fixed pieces would reach past the sequence)
    if (newL < base_len[w] || ((newL % PS) && refcount[row[newL / PS]] > 1)) {
        if (lane == 0) atomicExch(&counters[1], 4);
        return;
    }
    int freed = 0;
    for (int j = pages_of(newL) + lane; j < pages_of(L); j += 32) {
        const int p = row[j];
        row[j] = -1;
        if (atomicSub(&refcount[p], 1) == 1) ++freed;
    }
    for (int o = 16; o; o >>= 1) freed += __shfl_down_sync(0xffffffffu, freed, o);
    if (lane == 0) {
        if (freed) atomicAdd(&counters[0], freed);
        len[s] = newL;
    }
}

inline size_t al16(size_t x) { return (x + 15) & ~(size_t)15; }

bool turn_ok(const spork_turn *t) { return t && t->c && t->structure_epoch == t->c->structure_epoch; }

}  // namespace

extern "C" int spork_turn_prepare(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
                                  const int32_t *q_indptr, void *stream, spork_turn **out) {
    if (!c || !out || n_groups < 1 || !group_indptr || !seq_ids || !q_indptr || group_indptr[0] != 0 || q_indptr[0] != 0)
        return SPORK_ERR_INVALID;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    cudaStream_t st = (cudaStream_t)stream;
    const int n = group_indptr[n_groups];
    if (n < 1) return SPORK_ERR_INVALID;
    for (int i = 0; i < n; ++i) {
        const int s = seq_ids[i];
        if (s >= 0 && s < c->cfg.max_seqs) c->h_scratch[s] = 0;
    }
    for (int i = 0; i < n; ++i) {
        const int s = seq_ids[i], k = q_indptr[i + 1] - q_indptr[i];
        if (s < 0 || s >= c->cfg.max_seqs || !c->h_live[s] || c->h_scratch[s]++) return SPORK_ERR_INVALID_SEQ;
        if (k < 1 || k > 64 || c->h_len[s] < 1) return SPORK_ERR_INVALID;     // one block per request, <= 64 tokens
    }
    spork_turn *t = new (std::nothrow) spork_turn();
    if (!t) return SPORK_ERR_INVALID;
    t->c = c;
    t->n_seq = n;
    t->n_groups = n_groups;
    t->seq_ids.assign(seq_ids, seq_ids + n);
    t->group_indptr.assign(group_indptr, group_indptr + n_groups + 1);
    t->q_indptr.assign(q_indptr, q_indptr + n + 1);
    t->k.resize(n);
    t->base_len.resize(n);
    for (int i = 0; i < n; ++i) {
        t->k[i] = q_indptr[i + 1] - q_indptr[i];
        t->base_len[i] = c->h_len[seq_ids[i]];
        t->need_ub[0] += t->k[i] / PS + 1;
        t->need_ub[1] += 1;
        t->total_tok[0] += t->k[i];
        t->total_tok[1] += 1;
    }
    int rc = SPORK_OK;
    // ---- the two plans, built for the SHORTEST lengths their calls can meet (sequences only grow from turn
    // to turn: a turn nets accept_len + 1 >= 1 tokens): verify sees base + k, decode base + 1 ----
    Plan saved = std::move(c->plan);
    for (int which = 0; which < 2 && rc == SPORK_OK; ++which) {
        for (int i = 0; i < n; ++i) c->h_len[seq_ids[i]] = t->base_len[i] + (which == 0 ? t->k[i] : 1);
        c->plan = Plan();
        rc = build_plan(c, n_groups, group_indptr, seq_ids, which == 0 ? q_indptr : nullptr, st);
        if (rc == SPORK_OK && !c->plan.growable) rc = SPORK_ERR_INVALID;
        (which == 0 ? t->plan_v : t->plan_d) = std::move(c->plan);
    }
    for (int i = 0; i < n; ++i) c->h_len[seq_ids[i]] = t->base_len[i];
    c->plan = std::move(saved);
    // ---- descriptors that stay put on the device ----
    const size_t o_seq = 0, o_nt0 = al16(o_seq + 4 * (size_t)n), o_nt1 = al16(o_nt0 + 4 * (size_t)n);
    const size_t o_to0 = al16(o_nt1 + 4 * (size_t)n), o_to1 = al16(o_to0 + 4 * (size_t)n);
    const size_t o_base = al16(o_to1 + 4 * (size_t)n);
    const size_t o_qi = al16(o_base + 4 * (size_t)n), o_desc = al16(o_qi + 4 * (size_t)(n + 1));
    const size_t total = o_desc + sizeof(AppendDesc) * (size_t)n;
    if (rc == SPORK_OK) rc = devbuf_reserve(&t->dev, total, st);
    if (rc == SPORK_OK && (size_t)t->need_ub[0] > c->free_list_cap) {      // grow now: no reallocation under capture
        SPORK_CUDA(cudaStreamSynchronize(st));
        cudaFree(c->d_free_list);
        c->d_free_list = nullptr;
        c->free_list_cap = (size_t)t->need_ub[0] * 2;
        c->fl_valid = false;
        if (cudaMalloc(&c->d_free_list, c->free_list_cap * 4) != cudaSuccess) rc = SPORK_ERR_CUDA;
    }
    StageSlot *slot = nullptr;
    if (rc == SPORK_OK) rc = stage_acquire(c, o_desc, &slot);
    if (rc == SPORK_OK) {
        char *h = (char *)slot->h;
        int32_t *nt0 = (int32_t *)(h + o_nt0), *nt1 = (int32_t *)(h + o_nt1);
        int32_t *to0 = (int32_t *)(h + o_to0), *to1 = (int32_t *)(h + o_to1);
        memcpy(h + o_seq, seq_ids, 4 * (size_t)n);
        memcpy(h + o_base, t->base_len.data(), 4 * (size_t)n);
        memcpy(h + o_qi, q_indptr, 4 * (size_t)(n + 1));
        for (int i = 0; i < n; ++i) {
            nt0[i] = t->k[i];
            nt1[i] = 1;
            to0[i] = q_indptr[i];
            to1[i] = i;
        }
        if (cudaMemcpyAsync(t->dev.p, slot->h, o_desc, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = SPORK_ERR_CUDA;
        if (rc == SPORK_OK) rc = stage_done(c, slot, st);
    }
    if (rc != SPORK_OK) {
        spork_turn_destroy(t);
        return rc;
    }
    const char *d = (const char *)t->dev.p;
    t->d_seq = (const int32_t *)(d + o_seq);
    t->d_ntok[0] = (const int32_t *)(d + o_nt0);
    t->d_ntok[1] = (const int32_t *)(d + o_nt1);
    t->d_tokoff[0] = (const int32_t *)(d + o_to0);
    t->d_tokoff[1] = (const int32_t *)(d + o_to1);
    t->d_qi = (const int32_t *)(d + o_qi);
    t->d_base = (const int32_t *)(d + o_base);
    t->d_descs = (AppendDesc *)(d + o_desc);
    t->structure_epoch = c->structure_epoch;
    *out = t;
    return SPORK_OK;
}

extern "C" int spork_turn_destroy(spork_turn *t) {
    if (!t) return SPORK_OK;
    cudaDeviceSynchronize();
    for (DevBuf *b : {&t->dev, &t->plan_v.blob, &t->plan_d.blob})
        if (b->p) cudaFree(b->p);
    delete t;
    return SPORK_OK;
}

extern "C" int spork_turn_append(spork_turn *t, int which, const void *k_src, const void *v_src, void *stream) {
    if (!turn_ok(t) || which < 0 || which > 1 || !k_src || !v_src) return SPORK_ERR_INVALID;
    spork_ctx *c = t->c;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_launches = 0;
    c->mirror_stale = true;
    c->fl_valid = false;                   // the list is rebuilt by every call (how much of it a call uses is the device's secret)
    int rc = launch_free_scan(c, t->need_ub[which], st);
    if (rc != SPORK_OK) return rc;
    turn_append_plan_kernel<<<1, 256, 0, st>>>(t->d_seq, t->d_ntok[which], t->d_tokoff[which], t->n_seq, c->d_len,
                                               c->cfg.max_pages_per_seq, c->d_counters, t->d_descs);
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return launch_append_small(c, t->d_descs, t->n_seq, 0, k_src, v_src, st);
}

static int turn_attn(spork_turn *t, Plan &plan, const void *q, float *out, float *lse, cudaStream_t st) {
    if (!turn_ok(t)) return SPORK_ERR_INVALID;
    spork_ctx *c = t->c;
    c->last_launches = 0;
    std::swap(c->plan, plan);
    const LayerIO io{c->k_pool, c->v_pool, q, out, lse};
    const int rc = launch_planned(c, io, st);
    std::swap(c->plan, plan);
    return rc;
}

extern "C" int spork_turn_verify(spork_turn *t, const void *q, float *out, float *lse, void *stream) {
    return t ? turn_attn(t, t->plan_v, q, out, lse, (cudaStream_t)stream) : SPORK_ERR_INVALID;
}

extern "C" int spork_turn_decode(spork_turn *t, const void *q, float *out, float *lse, void *stream) {
    return t ? turn_attn(t, t->plan_d, q, out, lse, (cudaStream_t)stream) : SPORK_ERR_INVALID;
}

extern "C" int spork_turn_accept(spork_turn *t, const int32_t *draft_tokens, const int32_t *target_tokens,
                                 int32_t *accept_len_dev, void *stream) {
    if (!turn_ok(t) || !draft_tokens || !target_tokens) return SPORK_ERR_INVALID;
    spork_ctx *c = t->c;
    c->last_launches = 1;
    c->mirror_stale = true;
    c->fl_valid = false;
    turn_accept_kernel<<<ceil_div(t->n_seq, 4), 128, 0, (cudaStream_t)stream>>>(
        t->d_seq, t->d_qi, draft_tokens, target_tokens, t->d_base, t->n_seq, c->d_len, c->d_table, c->table_stride,
        c->d_refcount, c->d_counters, accept_len_dev);
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

// host mirror <- device: lengths of the turn's sequences, the free-page count; pages a sequence holds beyond
// what it held at spork_turn_prepare were allocated (possibly more than once) by the turns: its own
extern "C" int spork_turn_sync(spork_turn *t, void *stream) {
    if (!t || !t->c) return SPORK_ERR_INVALID;
    spork_ctx *c = t->c;
    SPORK_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    std::vector<int32_t> len((size_t)c->cfg.max_seqs);
    int32_t counters[2] = {0, 0};
    SPORK_CUDA(cudaMemcpy(len.data(), c->d_len, len.size() * 4, cudaMemcpyDeviceToHost));
    SPORK_CUDA(cudaMemcpy(counters, c->d_counters, 8, cudaMemcpyDeviceToHost));
    for (int i = 0; i < t->n_seq; ++i) {
        const int s = t->seq_ids[i];
        if (!c->h_live[s]) continue;
        if (len[s] != c->h_len[s]) {
            lineage_truncate(c, s, std::min(pages_of(t->base_len[i]), pages_of(len[s])));
            lineage_grow(c, s, pages_of(len[s]));
            c->h_shared_upto[s] = std::min(c->h_shared_upto[s], pages_of(len[s]));
        }
        c->h_len[s] = len[s];
    }
    c->free_lb = counters[0];
    c->fl_valid = false;
    c->len_epoch++;
    c->mirror_stale = false;
    return counters[1] == 0 ? SPORK_OK : SPORK_ERR_DEVICE;
}
