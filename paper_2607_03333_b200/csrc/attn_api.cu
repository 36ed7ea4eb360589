// libspork: spork_decode_attn / spork_verify_attn entry points.
#include "spork_internal.h"

using namespace spork;

static int attn_common(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
                       const int32_t *q_indptr, const void *q, float *out, float *lse,
                       cudaStream_t st) {
    c->last_launches = 0;
    int rc = build_plan(c, n_groups, group_indptr, seq_ids, q_indptr, st);
    if (rc != SPORK_OK) return rc;
    Plan &P = c->plan;
    if (P.n_qrows == 0) return SPORK_OK;
    if (!q || !out || !lse) return SPORK_ERR_INVALID;
    if (c->timing) SPORK_CUDA(cudaEventRecord(c->t_ev[0], st));
    if (P.info.kernel == 0) {
        rc = launch_attn_simt(c, q, st);
    } else {
        // longest streams first: the two-pipe tcgen05 kernel (items of > 128 rows), the one-pipe
        // tcgen05 kernel, then whatever the planner left to the mma.sync kernel.  A later kernel is
        // launched programmatically: it may start while the earlier one drains, and does not
        // complete before it (griddepcontrol.wait at its end), so the merge sees all partials.
        bool prev = false;
        rc = launch_attn_umma(c, q, 2, false, st);
        prev = P.n_items_umma2 > 0;
        if (rc == SPORK_OK) rc = launch_attn_umma(c, q, 1, prev, st);
        prev = prev || P.n_items_umma > 0;
        if (rc == SPORK_OK) rc = launch_attn_mma(c, q, prev, st);
    }
    if (rc != SPORK_OK) return rc;
    if (c->timing) SPORK_CUDA(cudaEventRecord(c->t_ev[1], st));
    if (P.info.kernel == 0) P.info.grid = P.n_items;
    if (P.info.kernel == 2) P.info.grid = P.grid_umma2 > 0 ? P.grid_umma2 : P.grid_umma;
    rc = launch_merge(c, out, lse, st);
    if (rc != SPORK_OK) return rc;
    if (c->timing) {
        SPORK_CUDA(cudaEventRecord(c->t_ev[2], st));
        c->t_valid = true;
    }
    P.info.launches = c->last_launches;
    SPORK_CUDA(cudaEventRecord(c->plan_ev, st));
    c->plan_ev_pending = true;
    return SPORK_OK;
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

static int attn_host(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
                     const int32_t *q_indptr, const void *q_host, float *out_host, float *lse_host,
                     cudaStream_t st) {
    if (n_groups < 0 || !group_indptr) return SPORK_ERR_INVALID;
    const int n_seq = group_indptr[n_groups];
    const size_t rows = q_indptr ? (size_t)q_indptr[n_seq] : (size_t)n_seq;
    const size_t Hq = c->cfg.num_q_heads, D = c->cfg.head_dim;
    const size_t qb = rows * Hq * D * c->elt, ob = rows * Hq * D * 4, lb = rows * Hq * 4;
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
