// libspork: handle lifetime, staging ring, sequence slots, synchronous export.
#include <string.h>

#include <algorithm>
#include <new>

#include "spork_internal.h"

using namespace spork;

// ---------------------------------------------------------------------------
// staging ring
// ---------------------------------------------------------------------------
namespace spork {

int stage_acquire(spork_ctx *c, size_t bytes, StageSlot **out) {
    StageSlot *s = &c->stage[c->stage_next];
    c->stage_next = (c->stage_next + 1) % 8;
    if (s->pending) {
        SPORK_CUDA(cudaEventSynchronize(s->ev));
        s->pending = false;
    }
    if (s->cap < bytes) {
        size_t cap = std::max<size_t>(bytes * 2, 1 << 16);
        if (s->h) cudaFreeHost(s->h);
        if (s->d) cudaFree(s->d);
        s->h = s->d = nullptr;
        s->cap = 0;
        SPORK_CUDA(cudaMallocHost(&s->h, cap));
        SPORK_CUDA(cudaMalloc(&s->d, cap));
        s->cap = cap;
    }
    if (!s->ev) SPORK_CUDA(cudaEventCreateWithFlags(&s->ev, cudaEventDisableTiming));
    *out = s;
    return SPORK_OK;
}

int stage_commit(spork_ctx *, StageSlot *s, size_t bytes, cudaStream_t st) {
    if (bytes) SPORK_CUDA(cudaMemcpyAsync(s->d, s->h, bytes, cudaMemcpyHostToDevice, st));
    return SPORK_OK;
}

int stage_done(spork_ctx *, StageSlot *s, cudaStream_t st) {
    SPORK_CUDA(cudaEventRecord(s->ev, st));
    s->pending = true;
    return SPORK_OK;
}

int devbuf_reserve(DevBuf *b, size_t bytes, cudaStream_t st) {
    if (b->cap >= bytes) return SPORK_OK;
    // growing is rare (first calls only): drain the stream, then reallocate
    SPORK_CUDA(cudaStreamSynchronize(st));
    if (b->p) cudaFree(b->p);
    b->p = nullptr;
    b->cap = 0;
    size_t cap = bytes + bytes / 4 + 4096;
    SPORK_CUDA(cudaMalloc(&b->p, cap));
    b->cap = cap;
    return SPORK_OK;
}

}  // namespace spork

// ---------------------------------------------------------------------------
// lifetime
// ---------------------------------------------------------------------------
extern "C" size_t spork_page_bytes(const spork_config *cfg) {
    if (!cfg) return 0;
    size_t elt = cfg->dtype == SPORK_F32 ? 4 : (cfg->dtype == SPORK_E4M3 ? 1 : 2);
    return (size_t)cfg->num_kv_heads * PS * cfg->head_dim * elt;
}

extern "C" const char *spork_strerror(int code) {
    switch (code) {
        case SPORK_OK: return "ok";
        case SPORK_ERR_INVALID: return "invalid argument";
        case SPORK_ERR_OOM: return "out of pages";
        case SPORK_ERR_NO_SLOT: return "out of sequence slots";
        case SPORK_ERR_TOO_LONG: return "sequence too long";
        case SPORK_ERR_INVALID_SEQ: return "invalid sequence id";
        case SPORK_ERR_SHARED: return "truncate into a shared partial page";
        case SPORK_ERR_CUDA: return "CUDA runtime error";
        case SPORK_ERR_DEVICE: return "device-side consistency check failed";
        case SPORK_ERR_STALE: return "host lengths are stale after a captured turn: call spork_turn_sync";
        case SPORK_ERR_LIMIT: return "size beyond the fixed maximum of a no-allocation entry point";
        default: return "unknown spork error";
    }
}

__global__ void init_state_kernel(int32_t *refcount, int num_pages, int32_t *table, size_t n_table,
                                  int32_t *len, int max_seqs, int32_t *counters) {
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t j = i; j < (size_t)num_pages; j += stride) refcount[j] = 0;
    for (size_t j = i; j < n_table; j += stride) table[j] = -1;
    for (size_t j = i; j < (size_t)max_seqs; j += stride) len[j] = 0;
    if (i == 0) {
        counters[0] = num_pages;
        for (int k = 1; k < 16; ++k) counters[k] = 0;
    }
}

extern "C" int spork_create(const spork_config *cfg, void *k_pool, void *v_pool, spork_ctx **out) {
    if (!cfg || !out || !k_pool || !v_pool) return SPORK_ERR_INVALID;
    if (cfg->dtype != SPORK_F32 && cfg->dtype != SPORK_BF16 && cfg->dtype != SPORK_E4M3) return SPORK_ERR_INVALID;
    if (cfg->num_q_heads <= 0 || cfg->num_kv_heads <= 0 || cfg->num_q_heads % cfg->num_kv_heads)
        return SPORK_ERR_INVALID;
    if (cfg->head_dim <= 0 || cfg->head_dim % 32 || cfg->head_dim > 256) return SPORK_ERR_INVALID;
    if (cfg->page_size != PS) return SPORK_ERR_INVALID;
    if (cfg->num_pages <= 0 || cfg->max_seqs <= 0 || cfg->max_pages_per_seq <= 0)
        return SPORK_ERR_INVALID;
    if (((uintptr_t)k_pool | (uintptr_t)v_pool) & 255) return SPORK_ERR_INVALID;

    spork_ctx *c = new (std::nothrow) spork_ctx();
    if (!c) return SPORK_ERR_INVALID;
    c->cfg = *cfg;
    c->G = cfg->num_q_heads / cfg->num_kv_heads;
    c->elt = cfg->dtype == SPORK_F32 ? 4 : (cfg->dtype == SPORK_E4M3 ? 1 : 2);
    c->q_elt = cfg->dtype == SPORK_F32 ? 4 : 2;
    c->swizzled = (cfg->dtype != SPORK_F32 && cfg->head_dim * c->elt % 128 == 0) ? 1 : 0;
    c->head_block = (size_t)PS * cfg->head_dim * c->elt;
    c->page_bytes = c->head_block * cfg->num_kv_heads;
    c->table_stride = (cfg->max_pages_per_seq + 3) & ~3;
    c->k_pool = k_pool;
    c->v_pool = v_pool;
    c->stage_next = 0;
    c->structure_epoch = 1;
    c->len_epoch = 1;
    c->free_lb = cfg->num_pages;
    c->n_live = 0;
    c->last_launches = 0;
    c->h_len.assign(cfg->max_seqs, 0);
    c->h_live.assign(cfg->max_seqs, 0);
    c->h_shared_upto.assign(cfg->max_seqs, 0);
    c->h_fork_key.assign(cfg->max_seqs, 0);
    c->h_fork_nf.assign(cfg->max_seqs, 0);
    c->h_scratch.assign(cfg->max_seqs, 0);
    c->h_lin.assign(cfg->max_seqs, Lineage{});
    c->h_uid.assign(cfg->max_seqs, 0);

    int dev = 0;
    bool ok = cudaGetDevice(&dev) == cudaSuccess &&
              cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess;
    size_t n_table = (size_t)cfg->max_seqs * c->table_stride;
    c->free_list_cap = 1 << 16;
    int scan_blocks = ceil_div(cfg->num_pages, 4096);
    ok = ok && cudaMalloc(&c->d_refcount, (size_t)cfg->num_pages * 4) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_table, n_table * 4) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_len, (size_t)cfg->max_seqs * 4) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_counters, 16 * 4) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_free_list, c->free_list_cap * 4) == cudaSuccess;
    ok = ok && cudaMalloc(&c->d_scan, (size_t)(scan_blocks + 1) * 4) == cudaSuccess;
    if (ok) {
        init_state_kernel<<<256, 256>>>(c->d_refcount, cfg->num_pages, c->d_table, n_table, c->d_len,
                                        cfg->max_seqs, c->d_counters);
        ok = cudaDeviceSynchronize() == cudaSuccess;
    }
    if (!ok) {
        spork_destroy(c);
        return SPORK_ERR_CUDA;
    }
    *out = c;
    return SPORK_OK;
}

extern "C" int spork_destroy(spork_ctx *c) {
    if (!c) return SPORK_OK;
    cudaDeviceSynchronize();
    cudaFree(c->d_refcount);
    cudaFree(c->d_table);
    cudaFree(c->d_len);
    cudaFree(c->d_counters);
    cudaFree(c->d_free_list);
    cudaFree(c->d_scan);
    for (auto &s : c->stage) {
        if (s.h) cudaFreeHost(s.h);
        if (s.d) cudaFree(s.d);
        if (s.ev) cudaEventDestroy(s.ev);
    }
    for (DevBuf *b : {&c->plan.blob, &c->ws_o, &c->ws_lse, &c->ws_conf, &c->conf_desc, &c->io_q, &c->io_out, &c->io_lse,
                      &c->d_layer_pools})
        if (b->p) cudaFree(b->p);
    for (auto &e : c->t_ev)
        if (e) cudaEventDestroy(e);
    delete c;
    return SPORK_OK;
}

// ---------------------------------------------------------------------------
// sequence slots (host bookkeeping; block tables and refcounts live on the device)
// ---------------------------------------------------------------------------
extern "C" int spork_seq_create(spork_ctx *c, int n, int32_t *ids_out) {
    if (!c || n < 0 || (n > 0 && !ids_out)) return SPORK_ERR_INVALID;
    if (c->cfg.max_seqs - c->n_live < n) return SPORK_ERR_NO_SLOT;
    for (int i = 0, s = 0; i < n; ++s)
        if (!c->h_live[s]) {
            c->h_live[s] = 1;
            c->h_len[s] = 0;
            c->h_shared_upto[s] = 0;
            c->h_fork_key[s] = 0;
            lineage_reset(c, s);
            ids_out[i++] = s;
        }
    c->n_live += n;
    c->structure_epoch++;
    c->len_epoch++;
    return SPORK_OK;
}

// ---------------------------------------------------------------------------
// synchronous export
// ---------------------------------------------------------------------------
extern "C" int spork_export(spork_ctx *c, int32_t seq, int32_t *len_out, int32_t *table_out) {
    if (!c || !len_out || seq < 0 || seq >= c->cfg.max_seqs) return SPORK_ERR_INVALID_SEQ;
    SPORK_CUDA(cudaDeviceSynchronize());
    if (!c->h_live[seq]) {
        *len_out = -1;
        return SPORK_OK;
    }
    int32_t dlen = 0;
    SPORK_CUDA(cudaMemcpy(&dlen, c->d_len + seq, 4, cudaMemcpyDeviceToHost));
    *len_out = dlen;  // the DEVICE length; tests compare it with the oracle's
    int np = pages_of(dlen);
    if (np > 0 && table_out)
        SPORK_CUDA(cudaMemcpy(table_out, c->d_table + (size_t)seq * c->table_stride, (size_t)np * 4,
                              cudaMemcpyDeviceToHost));
    return dlen == c->h_len[seq] ? SPORK_OK : SPORK_ERR_DEVICE;
}

extern "C" int spork_export_refcounts(spork_ctx *c, int32_t *host_out) {
    if (!c || !host_out) return SPORK_ERR_INVALID;
    SPORK_CUDA(cudaDeviceSynchronize());
    SPORK_CUDA(cudaMemcpy(host_out, c->d_refcount, (size_t)c->cfg.num_pages * 4,
                          cudaMemcpyDeviceToHost));
    return SPORK_OK;
}

extern "C" int spork_free_pages(spork_ctx *c, int32_t *out) {
    if (!c || !out) return SPORK_ERR_INVALID;
    SPORK_CUDA(cudaDeviceSynchronize());
    SPORK_CUDA(cudaMemcpy(out, c->d_counters, 4, cudaMemcpyDeviceToHost));
    c->free_lb = *out;
    return SPORK_OK;
}

extern "C" int spork_status(spork_ctx *c) {
    if (!c) return SPORK_ERR_INVALID;
    SPORK_CUDA(cudaDeviceSynchronize());
    int32_t e = 0;
    SPORK_CUDA(cudaMemcpy(&e, c->d_counters + 1, 4, cudaMemcpyDeviceToHost));
    return e == 0 ? SPORK_OK : SPORK_ERR_DEVICE;
}

extern "C" int spork_last_plan(spork_ctx *c, spork_plan_info *out) {
    if (!c || !out) return SPORK_ERR_INVALID;
    *out = c->plan.info;
    return SPORK_OK;
}

extern "C" int spork_last_launches(spork_ctx *c) { return c ? c->last_launches : SPORK_ERR_INVALID; }

// gather logical K/V rows out of the (possibly swizzled) pool
template <typename T>
__global__ void read_kv_kernel(const T *__restrict__ kpool, const T *__restrict__ vpool,
                               const int32_t *__restrict__ table_row, int t0, int n, int Hkv, int D,
                               int swizzled, T *__restrict__ k_out, T *__restrict__ v_out) {
    size_t total = (size_t)n * Hkv * D;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total;
         i += (size_t)gridDim.x * blockDim.x) {
        int d = (int)(i % D);
        int h = (int)((i / D) % Hkv);
        int t = t0 + (int)(i / ((size_t)D * Hkv));
        int page = table_row[t / PS];
        size_t off = ((size_t)page * Hkv + h) * (size_t)(PS * D) + head_block_off(swizzled, D, (int)sizeof(T), t % PS, d);
        k_out[i] = kpool[off];
        v_out[i] = vpool[off];
    }
}

extern "C" int spork_read_kv(spork_ctx *c, int32_t seq, int32_t t0, int32_t n, void *k_out,
                             void *v_out) {
    if (!c || seq < 0 || seq >= c->cfg.max_seqs || !c->h_live[seq]) return SPORK_ERR_INVALID_SEQ;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    if (t0 < 0 || n < 0 || t0 + n > c->h_len[seq] || (n > 0 && (!k_out || !v_out)))
        return SPORK_ERR_INVALID;
    if (n == 0) return SPORK_OK;
    SPORK_CUDA(cudaDeviceSynchronize());
    size_t bytes = (size_t)n * c->cfg.num_kv_heads * c->cfg.head_dim * c->elt;
    void *dk = nullptr, *dv = nullptr;
    SPORK_CUDA(cudaMalloc(&dk, bytes));
    if (cudaMalloc(&dv, bytes) != cudaSuccess) {
        cudaFree(dk);
        return SPORK_ERR_CUDA;
    }
    const int32_t *row = c->d_table + (size_t)seq * c->table_stride;
    if (c->elt == 4)
        read_kv_kernel<float><<<256, 256>>>((const float *)c->k_pool, (const float *)c->v_pool, row, t0,
                                            n, c->cfg.num_kv_heads, c->cfg.head_dim, c->swizzled,
                                            (float *)dk, (float *)dv);
    else if (c->elt == 1)
        read_kv_kernel<uint8_t><<<256, 256>>>((const uint8_t *)c->k_pool, (const uint8_t *)c->v_pool, row, t0,
                                              n, c->cfg.num_kv_heads, c->cfg.head_dim, c->swizzled,
                                              (uint8_t *)dk, (uint8_t *)dv);
    else
        read_kv_kernel<uint16_t><<<256, 256>>>((const uint16_t *)c->k_pool,
                                               (const uint16_t *)c->v_pool, row, t0, n,
                                               c->cfg.num_kv_heads, c->cfg.head_dim, c->swizzled,
                                               (uint16_t *)dk, (uint16_t *)dv);
    cudaError_t e = cudaMemcpy(k_out, dk, bytes, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(v_out, dv, bytes, cudaMemcpyDeviceToHost);
    cudaFree(dk);
    cudaFree(dv);
    return e == cudaSuccess ? SPORK_OK : SPORK_ERR_CUDA;
}
