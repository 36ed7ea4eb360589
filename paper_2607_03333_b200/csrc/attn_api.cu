// libspork: spork_decode_attn / spork_verify_attn entry points (single layer and multi-layer).
#include <string.h>

#include "spork_internal.h"

using namespace spork;

// One layer of the planned step: attention kernel(s), then the merge.  `chained`: this is layer > 0
// of a multi-layer call -- its first kernel is launched programmatically behind the previous layer's
// merge (which still reads the partial workspace: the kernel waits for it before its first partial).
static int launch_layer(spork_ctx *c, const LayerIO &io, bool chained, cudaStream_t st) {
    Plan &P = c->plan;
    int rc;
    if (P.info.kernel == 0) {
        rc = launch_attn_simt(c, io, st);
    } else {
        // longest streams first: the two-pipe tcgen05 kernel (items of > 128 rows), the one-pipe
        // tcgen05 kernel, then whatever the planner left to the mma.sync kernel.  A later kernel is
        // launched programmatically: it may start while the earlier one drains, and does not
        // complete before it (griddepcontrol.wait at its end), so the merge sees all partials.
        const bool pdl_chain = chained && P.info.kernel == 2;   // only the tcgen05 kernels know how to wait
        bool prev = false;
        rc = launch_attn_umma(c, io, 2, pdl_chain, pdl_chain, st);
        prev = P.n_items_umma2 > 0;
        if (rc == SPORK_OK) rc = launch_attn_umma(c, io, 1, prev || pdl_chain, pdl_chain, st);
        prev = prev || P.n_items_umma > 0;
        if (rc == SPORK_OK) rc = launch_attn_mma(c, io, prev, st);
    }
    return rc;
}

namespace spork {
int launch_planned(spork_ctx *c, const LayerIO &io, cudaStream_t st) {
    Plan &P = c->plan;
    if (!P.valid) return SPORK_ERR_INVALID;
    if (P.n_qrows == 0) return SPORK_OK;
    if (!io.q || !io.out || !io.lse) return SPORK_ERR_INVALID;
    int rc = launch_layer(c, io, false, st);
    if (rc == SPORK_OK) rc = launch_merge(c, io, st);
    return rc;
}
}  // namespace spork

static int attn_layers(spork_ctx *c, int n_layers, int n_groups, const int32_t *group_indptr,
                       const int32_t *seq_ids, const int32_t *q_indptr, const LayerIO *io, cudaStream_t st) {
    c->last_launches = 0;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    int rc = build_plan(c, n_groups, group_indptr, seq_ids, q_indptr, st);
    if (rc != SPORK_OK) return rc;
    Plan &P = c->plan;
    if (P.n_qrows == 0) return SPORK_OK;
    for (int l = 0; l < n_layers; ++l)
        if (!io[l].q || !io[l].out || !io[l].lse || !io[l].k_pool || !io[l].v_pool) return SPORK_ERR_INVALID;
    if (P.info.kernel == 0) P.info.grid = P.n_items;
    if (P.info.kernel == 2) P.info.grid = P.grid_umma2 > 0 ? P.grid_umma2 : P.grid_umma;
    for (int l = 0; l < n_layers; ++l) {
        const bool timed = c->timing && l == n_layers - 1;
        if (timed) SPORK_CUDA(cudaEventRecord(c->t_ev[0], st));
        rc = launch_layer(c, io[l], l > 0 && !c->timing, st);
        if (rc != SPORK_OK) return rc;
        if (timed) SPORK_CUDA(cudaEventRecord(c->t_ev[1], st));
        rc = launch_merge(c, io[l], st);
        if (rc != SPORK_OK) return rc;
        if (timed) {
            SPORK_CUDA(cudaEventRecord(c->t_ev[2], st));
            c->t_valid = true;
        }
    }
    P.info.launches = c->last_launches;
    return SPORK_OK;
}

static int attn_common(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
                       const int32_t *q_indptr, const void *q, float *out, float *lse,
                       cudaStream_t st) {
    const LayerIO io{c->k_pool, c->v_pool, q, out, lse};
    return attn_layers(c, 1, n_groups, group_indptr, seq_ids, q_indptr, &io, st);
}

extern "C" int spork_decode_attn(spork_ctx *c, int n_groups, const int32_t *group_indptr,
                                 const int32_t *seq_ids, const void *q, float *out, float *lse,
                                 void *stream) {
    if (!c) return SPORK_ERR_INVALID;
    return attn_common(c, n_groups, group_indptr, seq_ids, nullptr, q, out, lse, (cudaStream_t)stream);
}

extern "C" int spork_verify_attn(spork_ctx *c, int n_groups, const int32_t *group_indptr,
                                 const int32_t *seq_ids, const int32_t *q_indptr, const void *q,
                                 float *out, float *lse, void *stream) {
    if (!c || !q_indptr) return SPORK_ERR_INVALID;
    return attn_common(c, n_groups, group_indptr, seq_ids, q_indptr, q, out, lse, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------
// multi-layer step
// ---------------------------------------------------------------------------
extern "C" int spork_layers(spork_ctx *c, int n_layers, void *const *k_pools, void *const *v_pools, void *stream) {
    if (!c || n_layers < 1 || !k_pools || !v_pools) return SPORK_ERR_INVALID;
    if (k_pools[0] != c->k_pool || v_pools[0] != c->v_pool) return SPORK_ERR_INVALID;
    for (int l = 0; l < n_layers; ++l)
        if (!k_pools[l] || !v_pools[l] || (((uintptr_t)k_pools[l] | (uintptr_t)v_pools[l]) & 255)) return SPORK_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)stream;
    c->layer_k.assign(k_pools + 1, k_pools + n_layers);
    c->layer_v.assign(v_pools + 1, v_pools + n_layers);
    const size_t n = (size_t)(n_layers - 1);
    if (n) {
        int rc = devbuf_reserve(&c->d_layer_pools, 2 * n * sizeof(void *), st);
        if (rc != SPORK_OK) return rc;
        StageSlot *slot;
        rc = stage_acquire(c, 2 * n * sizeof(void *), &slot);
        if (rc != SPORK_OK) return rc;
        memcpy(slot->h, c->layer_k.data(), n * sizeof(void *));
        memcpy((char *)slot->h + n * sizeof(void *), c->layer_v.data(), n * sizeof(void *));
        SPORK_CUDA(cudaMemcpyAsync(c->d_layer_pools.p, slot->h, 2 * n * sizeof(void *), cudaMemcpyHostToDevice, st));
        rc = stage_done(c, slot, st);
        if (rc != SPORK_OK) return rc;
    }
    return SPORK_OK;
}

static int attn_layers_api(spork_ctx *c, int n_layers, int n_groups, const int32_t *group_indptr,
                           const int32_t *seq_ids, const int32_t *q_indptr, const void *const *q,
                           float *const *out, float *const *lse, cudaStream_t st) {
    if (!c || n_layers < 1 || n_layers > (int)c->layer_k.size() + 1 || !q || !out || !lse) return SPORK_ERR_INVALID;
    std::vector<LayerIO> io((size_t)n_layers);
    for (int l = 0; l < n_layers; ++l)
        io[l] = LayerIO{l == 0 ? c->k_pool : c->layer_k[l - 1], l == 0 ? c->v_pool : c->layer_v[l - 1], q[l], out[l], lse[l]};
    return attn_layers(c, n_layers, n_groups, group_indptr, seq_ids, q_indptr, io.data(), st);
}

extern "C" int spork_decode_attn_layers(spork_ctx *c, int n_layers, int n_groups, const int32_t *group_indptr,
                                        const int32_t *seq_ids, const void *const *q, float *const *out,
                                        float *const *lse, void *stream) {
    return attn_layers_api(c, n_layers, n_groups, group_indptr, seq_ids, nullptr, q, out, lse, (cudaStream_t)stream);
}

extern "C" int spork_verify_attn_layers(spork_ctx *c, int n_layers, int n_groups, const int32_t *group_indptr,
                                        const int32_t *seq_ids, const int32_t *q_indptr, const void *const *q,
                                        float *const *out, float *const *lse, void *stream) {
    if (!q_indptr) return SPORK_ERR_INVALID;
    return attn_layers_api(c, n_layers, n_groups, group_indptr, seq_ids, q_indptr, q, out, lse, (cudaStream_t)stream);
}

static int attn_host(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
                     const int32_t *q_indptr, const void *q_host, float *out_host, float *lse_host,
                     cudaStream_t st) {
    if (n_groups < 0 || !group_indptr) return SPORK_ERR_INVALID;
    const int n_seq = group_indptr[n_groups];
    const size_t rows = q_indptr ? (size_t)q_indptr[n_seq] : (size_t)n_seq;
    const size_t Hq = c->cfg.num_q_heads, D = c->cfg.head_dim;
    const size_t qb = rows * Hq * D * c->q_elt, ob = rows * Hq * D * 4, lb = rows * Hq * 4;
    if (rows == 0) return SPORK_OK;
    if (!q_host || !out_host || !lse_host) return SPORK_ERR_INVALID;
    int rc = devbuf_reserve(&c->io_q, qb, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&c->io_out, ob, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&c->io_lse, lb, st);
    if (rc != SPORK_OK) return rc;
    SPORK_CUDA(cudaMemcpyAsync(c->io_q.p, q_host, qb, cudaMemcpyHostToDevice, st));
    rc = attn_common(c, n_groups, group_indptr, seq_ids, q_indptr, c->io_q.p, (float *)c->io_out.p,
                     (float *)c->io_lse.p, st);
    if (rc != SPORK_OK) return rc;
    SPORK_CUDA(cudaMemcpyAsync(out_host, c->io_out.p, ob, cudaMemcpyDeviceToHost, st));
    SPORK_CUDA(cudaMemcpyAsync(lse_host, c->io_lse.p, lb, cudaMemcpyDeviceToHost, st));
    SPORK_CUDA(cudaStreamSynchronize(st));
    return SPORK_OK;
}

extern "C" int spork_decode_attn_host(spork_ctx *c, int n_groups, const int32_t *group_indptr,
                                      const int32_t *seq_ids, const void *q_host, float *out_host,
                                      float *lse_host, void *stream) {
    if (!c) return SPORK_ERR_INVALID;
    return attn_host(c, n_groups, group_indptr, seq_ids, nullptr, q_host, out_host, lse_host,
                     (cudaStream_t)stream);
}

extern "C" int spork_verify_attn_host(spork_ctx *c, int n_groups, const int32_t *group_indptr,
                                      const int32_t *seq_ids, const int32_t *q_indptr,
                                      const void *q_host, float *out_host, float *lse_host,
                                      void *stream) {
    if (!c || !q_indptr) return SPORK_ERR_INVALID;
    return attn_host(c, n_groups, group_indptr, seq_ids, q_indptr, q_host, out_host, lse_host,
                     (cudaStream_t)stream);
}

extern "C" int spork_set_timing(spork_ctx *c, int enable) {
    if (!c) return SPORK_ERR_INVALID;
    if (enable)
        for (auto &e : c->t_ev)
            if (!e) SPORK_CUDA(cudaEventCreate(&e));
    c->timing = enable ? 1 : 0;
    c->t_valid = false;
    return SPORK_OK;
}

extern "C" int spork_last_kernel_ms(spork_ctx *c, float *attn_ms, float *merge_ms) {
    if (!c || !attn_ms || !merge_ms || !c->t_valid) return SPORK_ERR_INVALID;
    SPORK_CUDA(cudaEventSynchronize(c->t_ev[2]));
    SPORK_CUDA(cudaEventElapsedTime(attn_ms, c->t_ev[0], c->t_ev[1]));
    SPORK_CUDA(cudaEventElapsedTime(merge_ms, c->t_ev[1], c->t_ev[2]));
    return SPORK_OK;
}

extern "C" int spork_set_tensor_path_min_rows(spork_ctx *c, int min_rows) {
    if (!c) return SPORK_ERR_INVALID;
    c->umma_min_rows = min_rows;
    c->plan.valid = false;
    return SPORK_OK;
}

extern "C" int spork_set_many_row_variant(spork_ctx *c, int enable) {
    if (!c) return SPORK_ERR_INVALID;
    c->many_row_variant = enable < 0 || enable > 2 ? 0 : enable;
    c->plan.valid = false;
    return SPORK_OK;
}

extern "C" int spork_set_stream_k(spork_ctx *c, int enable) {
    if (!c) return SPORK_ERR_INVALID;
    c->stream_k = enable ? 1 : 0;
    c->plan.valid = false;
    return SPORK_OK;
}

extern "C" int spork_set_cascade_levels(spork_ctx *c, int max_levels) {
    if (!c) return SPORK_ERR_INVALID;
    c->cascade_levels = max_levels < 1 ? 1 : (max_levels > MAX_ROW_REFS - 1 ? MAX_ROW_REFS - 1 : max_levels);
    c->plan.valid = false;
    return SPORK_OK;
}
