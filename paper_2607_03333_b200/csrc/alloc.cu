// libspork: page allocator (lowest free id first), append, fork, release, truncate.
//
// Device state: refcount[NP] (0 <=> free, reading A-2), table[S][stride],
// len[S], counters[0] = free pages.  The host mirrors only lengths and slot
// occupancy (to size grids and validate arguments); tables and refcounts are
// produced by these kernels alone.
#include <string.h>

#include <algorithm>
#include <unordered_map>

#include "spork_internal.h"

using namespace spork;

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_PER_THREAD = 16;
constexpr int SCAN_BLOCK = SCAN_THREADS * SCAN_PER_THREAD;  // 4096 pages per block

__device__ __forceinline__ int block_exclusive_scan(int v, int *total, int *smem /*[33]*/) {
    // 256 threads: warp scan + scan of the 8 warp totals
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) smem[w] = x;
    __syncthreads();
    if (w == 0) {
        int t = lane < (int)(blockDim.x >> 5) ? smem[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, t, o);
            if (lane >= o) t += y;
        }
        smem[lane] = t;  // inclusive warp totals
    }
    __syncthreads();
    int base = w ? smem[w - 1] : 0;
    *total = smem[(blockDim.x >> 5) - 1];
    return base + x - v;
}

// pass 1: number of free pages in each 4096-page block
__global__ void __launch_bounds__(SCAN_THREADS) free_count_kernel(const int32_t *__restrict__ refcount,
                                                                  int num_pages,
                                                                  int32_t *__restrict__ block_counts) {
    __shared__ int sm[33];
    int base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_PER_THREAD;
    int cnt = 0;
    if (base + SCAN_PER_THREAD <= num_pages) {
        const int4 *p = reinterpret_cast<const int4 *>(refcount + base);
#pragma unroll
        for (int i = 0; i < SCAN_PER_THREAD / 4; ++i) {
            int4 v = p[i];
            cnt += (v.x == 0) + (v.y == 0) + (v.z == 0) + (v.w == 0);
        }
    } else {
        for (int i = 0; i < SCAN_PER_THREAD; ++i)
            if (base + i < num_pages) cnt += refcount[base + i] == 0;
    }
    int total;
    block_exclusive_scan(cnt, &total, sm);
    if (threadIdx.x == 0) block_counts[blockIdx.x] = total;
}

// pass 2: exclusive scan of the block counts (single block, any length)
__global__ void __launch_bounds__(SCAN_THREADS) scan_blocks_kernel(int32_t *block_counts, int n) {
    __shared__ int sm[33];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int b = 0; b < n; b += SCAN_THREADS) {
        int i = b + threadIdx.x;
        int v = i < n ? block_counts[i] : 0;
        int total;
        int ex = block_exclusive_scan(v, &total, sm);
        int c0 = carry;
        if (i < n) block_counts[i] = c0 + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry = c0 + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) block_counts[n] = carry;  // total free pages
}

// pass 3: write the ids of the `need` lowest free pages, ascending
__global__ void __launch_bounds__(SCAN_THREADS) free_compact_kernel(
    const int32_t *__restrict__ refcount, int num_pages, const int32_t *__restrict__ block_offsets,
    int need, int32_t *__restrict__ free_list) {
    __shared__ int sm[33];
    int boff = block_offsets[blockIdx.x];
    if (boff >= need) return;
    int base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_PER_THREAD;
    unsigned mask = 0;
    if (base + SCAN_PER_THREAD <= num_pages) {
        const int4 *p = reinterpret_cast<const int4 *>(refcount + base);
#pragma unroll
        for (int i = 0; i < SCAN_PER_THREAD / 4; ++i) {
            int4 v = p[i];
            mask |= (unsigned)(v.x == 0) << (4 * i) | (unsigned)(v.y == 0) << (4 * i + 1) |
                    (unsigned)(v.z == 0) << (4 * i + 2) | (unsigned)(v.w == 0) << (4 * i + 3);
        }
    } else {
        for (int i = 0; i < SCAN_PER_THREAD; ++i)
            if (base + i < num_pages && refcount[base + i] == 0) mask |= 1u << i;
    }
    int total;
    int rank = boff + block_exclusive_scan(__popc(mask), &total, sm);
    while (mask && rank < need) {
        int i = __ffs(mask) - 1;
        mask &= mask - 1;
        free_list[rank++] = base + i;
    }
}

// ---- append (AppendDesc: spork_internal.h) -----------------------------------

__global__ void append_assign_kernel(const AppendDesc *__restrict__ descs, int n,
                                     const int32_t *__restrict__ free_list, int32_t *refcount,
                                     int32_t *table, int table_stride, int32_t *len, int32_t *counters,
                                     int need) {
    int i = blockIdx.x;
    AppendDesc d = descs[i];
    int first_new = pages_of(d.old_len);
    for (int j = threadIdx.x; j < d.n_new; j += blockDim.x) {
        int p = free_list[d.free_off + j];
        table[(size_t)d.seq * table_stride + first_new + j] = p;
        refcount[p] = 1;
    }
    if (threadIdx.x == 0) {
        if (d.final_len >= 0) len[d.seq] = d.final_len;
        if (i == 0 && need) atomicSub(&counters[0], need);
    }
}

// one thread per 16-byte chunk of one (token, kv head) row; K and V together
__global__ void __launch_bounds__(256) append_copy_kernel(
    const AppendDesc *__restrict__ descs, int n, const uint4 *__restrict__ k_src,
    const uint4 *__restrict__ v_src, uint8_t *__restrict__ k_pool, uint8_t *__restrict__ v_pool,
    const int32_t *__restrict__ table, int table_stride, int Hkv, int chunks_per_row /* D*elt/16 */,
    int swizzled, size_t head_block, size_t total_units) {
    for (size_t u = blockIdx.x * (size_t)blockDim.x + threadIdx.x; u < total_units;
         u += (size_t)gridDim.x * blockDim.x) {
        int c = (int)(u % chunks_per_row);
        int h = (int)((u / chunks_per_row) % Hkv);
        int tok = (int)(u / ((size_t)chunks_per_row * Hkv));
        // request containing flat token `tok`: last i with tok_off <= tok
        int lo = 0, hi = n - 1;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (descs[mid].tok_off <= tok) lo = mid; else hi = mid - 1;
        }
        // requests with n_tok == 0 share tok_off with their successor: the search lands on the last
        // of them, which is the one that owns the token
        AppendDesc d = descs[lo];
        int pos = d.old_len + (tok - d.tok_off);
        int page = table[(size_t)d.seq * table_stride + pos / PS];
        int r = pos % PS;
        size_t off;
        if (swizzled) {
            off = (size_t)swz_chunk_off(chunks_per_row >> 3, r, c);
        } else {
            off = ((size_t)r * chunks_per_row + c) * 16;
        }
        size_t dst = ((size_t)page * Hkv + h) * head_block + off;
        *reinterpret_cast<uint4 *>(k_pool + dst) = k_src[u];
        *reinterpret_cast<uint4 *>(v_pool + dst) = v_src[u];
    }
}

// The decode loop's append (Algorithm 1 step 5: one token per live stream and step): few tokens per
// request and no sequence twice in the batch -> ONE kernel, one block per request: take the pages,
// publish the length, then write this request's K/V rows (its table entries are its own block's).
__device__ __forceinline__ void append_small_body(
    const AppendDesc d, const int32_t *__restrict__ free_list, int32_t *refcount,
    int32_t *table, int table_stride, int32_t *len, int32_t *counters, int need,
    const uint4 *__restrict__ k_src, const uint4 *__restrict__ v_src, uint8_t *__restrict__ k_pool,
    uint8_t *__restrict__ v_pool, int Hkv, int chunks_per_row, int swizzled, size_t head_block) {
    __shared__ int32_t s_page[8];                 // pages of positions old_len .. (<= 64 tokens: <= 5 pages)
    int32_t *row = table + (size_t)d.seq * table_stride;
    const int first_new = pages_of(d.old_len), p0 = d.old_len / PS;
    const int n_touch = d.n_tok > 0 ? (d.old_len + d.n_tok - 1) / PS - p0 + 1 : 0;
    if ((int)threadIdx.x < n_touch) {
        const int j = p0 + threadIdx.x;
        int p;
        if (j >= first_new) {
            p = free_list[d.free_off + (j - first_new)];
            row[j] = p;
            refcount[p] = 1;
        } else {
            p = row[j];                           // the partially filled tail page it already holds
        }
        s_page[threadIdx.x] = p;
    }
    if (threadIdx.x == 0) {
        if (d.final_len >= 0) len[d.seq] = d.final_len;
        if (blockIdx.x == 0 && need) atomicSub(&counters[0], need);
    }
    __syncthreads();
    const int units = d.n_tok * Hkv * chunks_per_row;
    for (int u = threadIdx.x; u < units; u += blockDim.x) {
        const int c = u % chunks_per_row, h = (u / chunks_per_row) % Hkv, t = u / (chunks_per_row * Hkv);
        const int pos = d.old_len + t, r = pos % PS;
        const size_t off = swizzled ? (size_t)swz_chunk_off(chunks_per_row >> 3, r, c)
                                    : ((size_t)r * chunks_per_row + c) * 16;
        const size_t dst = ((size_t)s_page[pos / PS - p0] * Hkv + h) * head_block + off;
        const size_t src = (size_t)d.tok_off * Hkv * chunks_per_row + u;
        *reinterpret_cast<uint4 *>(k_pool + dst) = k_src[src];
        *reinterpret_cast<uint4 *>(v_pool + dst) = v_src[src];
    }
}

__global__ void __launch_bounds__(128) append_small_kernel(
    const AppendDesc *__restrict__ descs, const int32_t *__restrict__ free_list, int32_t *refcount,
    int32_t *table, int table_stride, int32_t *len, int32_t *counters, int need,
    const uint4 *__restrict__ k_src, const uint4 *__restrict__ v_src, uint8_t *__restrict__ k_pool,
    uint8_t *__restrict__ v_pool, int Hkv, int chunks_per_row, int swizzled, size_t head_block) {
    append_small_body(descs[blockIdx.x], free_list, refcount, table, table_stride, len, counters, need, k_src, v_src,
                      k_pool, v_pool, Hkv, chunks_per_row, swizzled, head_block);
}

// the same with the descriptors of a small batch passed as kernel PARAMETERS: the decode loop's append needs
// no host-to-device copy at all (one launch; 3 us of a 12 us call)
constexpr int APPEND_PARAM_MAX = 96;              // 96 x 32 B = 3 KiB of the 4 KiB parameter space
struct AppendDescPack {
    AppendDesc d[APPEND_PARAM_MAX];
};
__global__ void __launch_bounds__(128) append_small_param_kernel(
    const __grid_constant__ AppendDescPack pack, const int32_t *__restrict__ free_list, int32_t *refcount,
    int32_t *table, int table_stride, int32_t *len, int32_t *counters, int need,
    const uint4 *__restrict__ k_src, const uint4 *__restrict__ v_src, uint8_t *__restrict__ k_pool,
    uint8_t *__restrict__ v_pool, int Hkv, int chunks_per_row, int swizzled, size_t head_block) {
    append_small_body(pack.d[blockIdx.x], free_list, refcount, table, table_stride, len, counters, need, k_src, v_src,
                      k_pool, v_pool, Hkv, chunks_per_row, swizzled, head_block);
}

// ---- fork ------------------------------------------------------------------
struct ForkDesc {
    int32_t parent, child, len, tail_idx;  // tail_idx: index into free_list, or -1
};
struct ParentDesc {
    int32_t parent, count, nf, pad;
};

// one block per fork: clone the table row (16-byte vectors), then duplicate the tail page
__global__ void __launch_bounds__(256) fork_clone_kernel(
    const ForkDesc *__restrict__ descs, const int32_t *__restrict__ free_list, int32_t *table,
    int table_stride, int32_t *len, int32_t *refcount, uint8_t *k_pool, uint8_t *v_pool,
    size_t page_bytes, int32_t *counters, int need, int n_extra_pools, uint8_t *const *extra_pools) {
    __shared__ int s_tail;
    ForkDesc d = descs[blockIdx.x];
    int nf = d.len / PS;
    int tail_page = d.tail_idx >= 0 ? free_list[d.tail_idx] : -1;
    const int4 *src = reinterpret_cast<const int4 *>(table + (size_t)d.parent * table_stride);
    int4 *dst = reinterpret_cast<int4 *>(table + (size_t)d.child * table_stride);
    int n4 = (nf + 1 + 3) / 4;                       // covers entries [0, nf]
    if (n4 * 4 > table_stride) n4 = table_stride / 4;
    int parent_tail = -1;
    for (int j = threadIdx.x; j < n4; j += blockDim.x) {
        int4 v = src[j];
        int e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            int idx = j * 4 + q;
            if (idx == nf) { parent_tail = e[q]; e[q] = tail_page; }
            else if (idx > nf) e[q] = -1;
        }
        dst[j] = make_int4(e[0], e[1], e[2], e[3]);
    }
    if (threadIdx.x == 0) {
        len[d.child] = d.len;
        if (tail_page >= 0) refcount[tail_page] = 1;
        if (blockIdx.x == 0 && need) atomicSub(&counters[0], need);
    }
    if (tail_page < 0) return;
    // the thread that saw entry nf broadcasts the parent's tail page id
    if (parent_tail >= 0) s_tail = parent_tail;
    __syncthreads();
    size_t n16 = page_bytes / 16;
    const uint4 *ks = reinterpret_cast<const uint4 *>(k_pool + (size_t)s_tail * page_bytes);
    const uint4 *vs = reinterpret_cast<const uint4 *>(v_pool + (size_t)s_tail * page_bytes);
    uint4 *kd = reinterpret_cast<uint4 *>(k_pool + (size_t)tail_page * page_bytes);
    uint4 *vd = reinterpret_cast<uint4 *>(v_pool + (size_t)tail_page * page_bytes);
    for (size_t j = threadIdx.x; j < n16; j += blockDim.x) {
        kd[j] = ks[j];
        vd[j] = vs[j];
    }
    // the other layers' pools (spork_layers): block tables are shared, so the tail is duplicated in each
    for (int e = 0; e < n_extra_pools; ++e) {
        const uint4 *src2 = reinterpret_cast<const uint4 *>(extra_pools[e] + (size_t)s_tail * page_bytes);
        uint4 *dst2 = reinterpret_cast<uint4 *>(extra_pools[e] + (size_t)tail_page * page_bytes);
        for (size_t j = threadIdx.x; j < n16; j += blockDim.x) dst2[j] = src2[j];
    }
}

// one block per (distinct parent, 1024-entry chunk): refcount[page] += number of forks of that parent
__global__ void __launch_bounds__(256) fork_refcount_kernel(const ParentDesc *__restrict__ pd,
                                                            const int32_t *__restrict__ table,
                                                            int table_stride, int32_t *refcount) {
    ParentDesc d = pd[blockIdx.y];
    const int32_t *row = table + (size_t)d.parent * table_stride;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < d.nf; j += gridDim.x * blockDim.x)
        atomicAdd(&refcount[row[j]], d.count);
}

// ---- release / truncate ------------------------------------------------------
struct DropDesc {
    int32_t seq, keep_pages, n_pages, new_len;
    // release of several children of one fork (same parent, same call): their first agg_upto table
    // entries are the same pages.  The first of them in the request subtracts the whole family's
    // references at once (agg_mult = family size), the others skip those pages (agg_mult = 0):
    // 10k releases of 128 families are 0.3 M atomics on the hot pages instead of 21.8 M.
    int32_t agg_upto, agg_mult;
};

// one block per sequence: drop its references from pages [keep_pages, n_pages)
__global__ void __launch_bounds__(256) drop_pages_kernel(const DropDesc *__restrict__ descs,
                                                         int32_t *table, int table_stride,
                                                         int32_t *len, int32_t *refcount,
                                                         int32_t *counters) {
    __shared__ int s_freed;
    DropDesc d = descs[blockIdx.x];
    if (threadIdx.x == 0) s_freed = 0;
    __syncthreads();
    int32_t *row = table + (size_t)d.seq * table_stride;
    int freed = 0;
    // 4 table entries per thread are loaded before the first store / atomic (which the compiler must
    // keep in order with later loads of the same array): one memory round trip per 1,024 pages
    for (int j0 = d.keep_pages + threadIdx.x; j0 < d.n_pages; j0 += 4 * blockDim.x) {
        int p[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = j0 + u * blockDim.x;
            p[u] = j < d.n_pages ? __ldcg(row + j) : -2;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = j0 + u * blockDim.x;
            if (p[u] == -2) continue;
            row[j] = -1;
            if (p[u] < 0) { atomicExch(&counters[1], 1); continue; }   // consistency check
            const int mult = j < d.agg_upto ? d.agg_mult : 1;
            if (mult == 0) continue;                                   // the family's leader drops these
            int old = atomicSub(&refcount[p[u]], mult);
            if (old == mult) ++freed;
            if (old < mult) atomicExch(&counters[1], 2);
        }
    }
    for (int o = 16; o; o >>= 1) freed += __shfl_down_sync(0xffffffffu, freed, o);
    if ((threadIdx.x & 31) == 0 && freed) atomicAdd(&s_freed, freed);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_freed) atomicAdd(&counters[0], s_freed);
        len[d.seq] = d.new_len;
    }
}

__global__ void check_shared_kernel(const DropDesc *__restrict__ descs, int n,
                                    const int32_t *__restrict__ table, int table_stride,
                                    const int32_t *__restrict__ refcount, int32_t *flag) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        DropDesc d = descs[i];
        if (d.new_len % PS) {
            int p = table[(size_t)d.seq * table_stride + d.new_len / PS];
            if (p < 0 || refcount[p] > 1) *flag = 1;
        }
    }
}

}  // namespace

// ---------------------------------------------------------------------------
namespace spork {

int launch_free_scan(spork_ctx *c, int need, cudaStream_t st) {
    if (need <= 0) return SPORK_OK;
    if ((size_t)need > c->free_list_cap) {
        SPORK_CUDA(cudaStreamSynchronize(st));
        cudaFree(c->d_free_list);
        c->d_free_list = nullptr;
        c->free_list_cap = (size_t)need * 2;
        SPORK_CUDA(cudaMalloc(&c->d_free_list, c->free_list_cap * 4));
    }
    int nb = ceil_div(c->cfg.num_pages, SCAN_BLOCK);
    free_count_kernel<<<nb, SCAN_THREADS, 0, st>>>(c->d_refcount, c->cfg.num_pages, c->d_scan);
    scan_blocks_kernel<<<1, SCAN_THREADS, 0, st>>>(c->d_scan, nb);
    free_compact_kernel<<<nb, SCAN_THREADS, 0, st>>>(c->d_refcount, c->cfg.num_pages, c->d_scan, need,
                                                     c->d_free_list);
    c->last_launches += 3;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

int ensure_pages(spork_ctx *c, int64_t need, cudaStream_t st) {
    if (need <= c->free_lb) return SPORK_OK;
    // the lower bound cannot prove it: read the exact device count (documented sync)
    SPORK_CUDA(cudaStreamSynchronize(st));
    int32_t f = 0;
    SPORK_CUDA(cudaMemcpy(&f, c->d_counters, 4, cudaMemcpyDeviceToHost));
    c->free_lb = f;
    return need <= c->free_lb ? SPORK_OK : SPORK_ERR_OOM;
}

// the one-kernel append over descriptors that are already on the device (spork_append's fast path; turn.cu)
int launch_append_small(spork_ctx *c, const AppendDesc *d_descs, int n, int need, const void *k_src,
                        const void *v_src, cudaStream_t st) {
    append_small_kernel<<<n, 128, 0, st>>>(
        d_descs, c->d_free_list, c->d_refcount, c->d_table, c->table_stride, c->d_len, c->d_counters, need,
        (const uint4 *)k_src, (const uint4 *)v_src, (uint8_t *)c->k_pool, (uint8_t *)c->v_pool,
        c->cfg.num_kv_heads, c->cfg.head_dim * c->elt / 16, c->swizzled, c->head_block);
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

// `need` lowest free page ids, ascending, at d_free_list[*off ..).  The list of one scan is cached: as long
// as no page has been FREED since (release / truncate / accept invalidate it), the ids behind the ones
// already handed out are still the lowest free ones, so an append-only phase (the decode loop) scans
// once per FREE_LIST_BATCH pages instead of once per call.
int take_free(spork_ctx *c, int need, cudaStream_t st, int *off) {
    *off = 0;
    if (need <= 0) return SPORK_OK;
    if (c->fl_valid && c->fl_pos + need <= c->fl_n) {
        *off = c->fl_pos;
        c->fl_pos += need;
        return SPORK_OK;
    }
    // free_lb is a lower bound on the free pages (ensure_pages has run): every id of the list is real
    constexpr int64_t FREE_LIST_BATCH = 4096;
    const int want = (int)std::max<int64_t>(need, std::min<int64_t>(c->free_lb, FREE_LIST_BATCH));
    int rc = launch_free_scan(c, want, st);
    if (rc != SPORK_OK) return rc;
    c->fl_valid = true;
    c->fl_n = want;
    c->fl_pos = need;
    return SPORK_OK;
}

}  // namespace spork

// ---------------------------------------------------------------------------
extern "C" int spork_append(spork_ctx *c, int n, const int32_t *seq_ids, const int32_t *n_tokens,
                            const void *k_src, const void *v_src, void *stream) {
    if (!c || n < 0 || (n > 0 && (!seq_ids || !n_tokens))) return SPORK_ERR_INVALID;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_launches = 0;
    if (n == 0) return SPORK_OK;
    // validate the whole batch against evolving lengths; nothing changes on failure
    for (int i = 0; i < n; ++i) {
        int s = seq_ids[i];
        if (s >= 0 && s < c->cfg.max_seqs && c->h_live[s]) c->h_scratch[s] = c->h_len[s];
    }
    int64_t need = 0, total = 0;
    for (int i = 0; i < n; ++i) {
        int s = seq_ids[i];
        if (s < 0 || s >= c->cfg.max_seqs || !c->h_live[s] || n_tokens[i] < 0)
            return SPORK_ERR_INVALID_SEQ;
        int64_t nl = (int64_t)c->h_scratch[s] + n_tokens[i];
        if ((nl + PS - 1) / PS > c->cfg.max_pages_per_seq) return SPORK_ERR_TOO_LONG;
        need += pages_of((int)nl) - pages_of(c->h_scratch[s]);
        c->h_scratch[s] = (int)nl;
        total += n_tokens[i];
    }
    if (total > 0 && (!k_src || !v_src)) return SPORK_ERR_INVALID;
    if (total >= (int64_t)1 << 31) return SPORK_ERR_INVALID;
    int rc = ensure_pages(c, need, st);
    if (rc != SPORK_OK) return rc;

    // a small batch (the decode loop) carries its descriptors in the kernel parameters; others stage them
    AppendDescPack pack;
    StageSlot *slot = nullptr;
    AppendDesc *d = pack.d;
    if (n > APPEND_PARAM_MAX) {
        rc = stage_acquire(c, sizeof(AppendDesc) * (size_t)n, &slot);
        if (rc != SPORK_OK) return rc;
        d = (AppendDesc *)slot->h;
    }
    for (int i = 0; i < n; ++i) c->h_scratch[seq_ids[i]] = -1;  // marks "last request not yet seen"
    int fl_off = 0;
    rc = take_free(c, (int)need, st, &fl_off);
    if (rc != SPORK_OK) return rc;
    int tok = 0, foff = fl_off;
    bool small = true;       // no sequence twice, <= 64 tokens per request: the one-kernel path
    // final_len is written by the LAST request of each sequence: walk backwards to mark it
    for (int i = n - 1; i >= 0; --i) {
        int s = seq_ids[i];
        d[i].final_len = c->h_scratch[s] == -1 ? 0 : -1;  // placeholder 0 = "is last"
        small = small && c->h_scratch[s] == -1 && n_tokens[i] <= 64;
        c->h_scratch[s] = 0;
    }
    for (int i = 0; i < n; ++i) {
        int s = seq_ids[i];
        int ol = c->h_len[s], nl = ol + n_tokens[i];
        d[i].seq = s;
        d[i].old_len = ol;
        d[i].n_tok = n_tokens[i];
        d[i].tok_off = tok;
        d[i].free_off = foff;
        d[i].n_new = pages_of(nl) - pages_of(ol);
        d[i].final_len = d[i].final_len == 0 ? nl : -1;
        d[i].pad = 0;
        tok += n_tokens[i];
        foff += d[i].n_new;
        c->h_len[s] = nl;
        lineage_grow(c, s, pages_of(nl));
    }
    if (small && !slot) {
        append_small_param_kernel<<<n, 128, 0, st>>>(
            pack, c->d_free_list, c->d_refcount, c->d_table, c->table_stride, c->d_len, c->d_counters, (int)need,
            (const uint4 *)k_src, (const uint4 *)v_src, (uint8_t *)c->k_pool, (uint8_t *)c->v_pool,
            c->cfg.num_kv_heads, c->cfg.head_dim * c->elt / 16, c->swizzled, c->head_block);
        c->last_launches++;
        SPORK_CUDA(cudaGetLastError());
        c->free_lb -= need;
        c->len_epoch++;
        return SPORK_OK;
    }
    if (!slot) {        // few requests but not the one-kernel shape (a repeated sequence, a long request): stage after all
        rc = stage_acquire(c, sizeof(AppendDesc) * (size_t)n, &slot);
        if (rc != SPORK_OK) return rc;
        memcpy(slot->h, pack.d, sizeof(AppendDesc) * (size_t)n);
    }
    rc = stage_commit(c, slot, sizeof(AppendDesc) * (size_t)n, st);
    if (rc != SPORK_OK) return rc;
    if (small) {
        rc = launch_append_small(c, (const AppendDesc *)slot->d, n, (int)need, k_src, v_src, st);
        if (rc != SPORK_OK) return rc;
        c->free_lb -= need;
        c->len_epoch++;
        return stage_done(c, slot, st);
    }
    append_assign_kernel<<<n, 128, 0, st>>>((const AppendDesc *)slot->d, n, c->d_free_list,
                                            c->d_refcount, c->d_table, c->table_stride, c->d_len,
                                            c->d_counters, (int)need);
    c->last_launches++;
    if (total > 0) {
        int cpr = c->cfg.head_dim * c->elt / 16;
        size_t units = (size_t)total * c->cfg.num_kv_heads * cpr;
        int blocks = (int)std::min<size_t>((units + 255) / 256, (size_t)c->num_sms * 16);
        append_copy_kernel<<<blocks, 256, 0, st>>>(
            (const AppendDesc *)slot->d, n, (const uint4 *)k_src, (const uint4 *)v_src,
            (uint8_t *)c->k_pool, (uint8_t *)c->v_pool, c->d_table, c->table_stride,
            c->cfg.num_kv_heads, cpr, c->swizzled, c->head_block, units);
        c->last_launches++;
    }
    SPORK_CUDA(cudaGetLastError());
    c->free_lb -= need;
    c->len_epoch++;
    return stage_done(c, slot, st);
}

// K/V of the LAST n_tokens[i] tokens of each sequence into another layer's pools:
// the pages were allocated by spork_append (block tables are shared by all layers)
extern "C" int spork_write_kv_layer(spork_ctx *c, int layer, int n, const int32_t *seq_ids,
                                    const int32_t *n_tokens, const void *k_src, const void *v_src, void *stream) {
    if (!c || n < 0 || (n > 0 && (!seq_ids || !n_tokens))) return SPORK_ERR_INVALID;
    if (layer < 0 || layer > (int)c->layer_k.size()) return SPORK_ERR_INVALID;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_launches = 0;
    if (n == 0) return SPORK_OK;
    int64_t total = 0;
    for (int i = 0; i < n; ++i) {
        const int s = seq_ids[i];
        if (s < 0 || s >= c->cfg.max_seqs || !c->h_live[s]) return SPORK_ERR_INVALID_SEQ;
        if (n_tokens[i] < 0 || n_tokens[i] > c->h_len[s]) return SPORK_ERR_INVALID;
        total += n_tokens[i];
    }
    if (total == 0) return SPORK_OK;
    if (!k_src || !v_src || total >= (int64_t)1 << 31) return SPORK_ERR_INVALID;
    StageSlot *slot;
    int rc = stage_acquire(c, sizeof(AppendDesc) * (size_t)n, &slot);
    if (rc != SPORK_OK) return rc;
    AppendDesc *d = (AppendDesc *)slot->h;
    int tok = 0;
    for (int i = 0; i < n; ++i) {
        d[i] = AppendDesc{seq_ids[i], c->h_len[seq_ids[i]] - n_tokens[i], n_tokens[i], tok, 0, 0, -1, 0};
        tok += n_tokens[i];
    }
    rc = stage_commit(c, slot, sizeof(AppendDesc) * (size_t)n, st);
    if (rc != SPORK_OK) return rc;
    const int cpr = c->cfg.head_dim * c->elt / 16;
    const size_t units = (size_t)total * c->cfg.num_kv_heads * cpr;
    const int blocks = (int)std::min<size_t>((units + 255) / 256, (size_t)c->num_sms * 16);
    uint8_t *kp = (uint8_t *)(layer == 0 ? c->k_pool : c->layer_k[layer - 1]);
    uint8_t *vp = (uint8_t *)(layer == 0 ? c->v_pool : c->layer_v[layer - 1]);
    append_copy_kernel<<<blocks, 256, 0, st>>>((const AppendDesc *)slot->d, n, (const uint4 *)k_src,
                                               (const uint4 *)v_src, kp, vp, c->d_table, c->table_stride,
                                               c->cfg.num_kv_heads, cpr, c->swizzled, c->head_block, units);
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return stage_done(c, slot, st);
}

extern "C" int spork_fork(spork_ctx *c, int n, const int32_t *parent_ids, int32_t *child_ids_out,
                          void *stream) {
    if (!c || n < 0 || (n > 0 && (!parent_ids || !child_ids_out))) return SPORK_ERR_INVALID;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_launches = 0;
    if (n == 0) return SPORK_OK;
    int64_t need = 0;
    for (int i = 0; i < n; ++i) {
        int p = parent_ids[i];
        if (p < 0 || p >= c->cfg.max_seqs || !c->h_live[p]) return SPORK_ERR_INVALID_SEQ;
        need += (c->h_len[p] % PS) != 0;
    }
    if (c->cfg.max_seqs - c->n_live < n) return SPORK_ERR_NO_SLOT;
    int rc = ensure_pages(c, need, st);
    if (rc != SPORK_OK) return rc;

    size_t bytes = sizeof(ForkDesc) * (size_t)n + sizeof(ParentDesc) * (size_t)n;
    StageSlot *slot;
    rc = stage_acquire(c, bytes, &slot);
    if (rc != SPORK_OK) return rc;
    ForkDesc *fd = (ForkDesc *)slot->h;
    ParentDesc *pd = (ParentDesc *)(fd + n);
    // count forks per distinct parent (h_scratch as a per-slot counter)
    for (int i = 0; i < n; ++i) c->h_scratch[parent_ids[i]] = 0;
    int n_par = 0, max_nf = 0;
    for (int i = 0; i < n; ++i) {
        int p = parent_ids[i];
        if (c->h_scratch[p]++ == 0) {
            pd[n_par].parent = p;
            pd[n_par].nf = c->h_len[p] / PS;
            pd[n_par].pad = 0;
            max_nf = std::max(max_nf, pd[n_par].nf);
            ++n_par;
        }
    }
    for (int j = 0; j < n_par; ++j) pd[j].count = c->h_scratch[pd[j].parent];
    // children: lowest free slots in request order
    c->fork_calls++;
    int tail = 0;
    rc = take_free(c, (int)need, st, &tail);
    if (rc != SPORK_OK) return rc;
    for (int i = 0, s = 0; i < n; ++s) {
        if (c->h_live[s]) continue;
        int p = parent_ids[i], L = c->h_len[p];
        c->h_live[s] = 1;
        c->h_len[s] = L;
        c->h_shared_upto[s] = L / PS;
        c->h_shared_upto[p] = std::max(c->h_shared_upto[p], L / PS);
        c->h_fork_key[s] = (c->fork_calls << 32) | (uint64_t)(p + 1);   // same call, same parent: same prefix
        c->h_fork_nf[s] = L / PS;
        lineage_fork(c, s, p, L);
        fd[i].parent = p;
        fd[i].child = s;
        fd[i].len = L;
        fd[i].tail_idx = (L % PS) ? tail++ : -1;
        child_ids_out[i] = s;
        ++i;
    }
    c->n_live += n;
    rc = stage_commit(c, slot, bytes, st);
    if (rc != SPORK_OK) return rc;
    if (max_nf > 0) {
        dim3 grid(std::max(1, std::min(ceil_div(max_nf, 1024), 64)), n_par);
        fork_refcount_kernel<<<grid, 256, 0, st>>>((const ParentDesc *)((ForkDesc *)slot->d + n),
                                                   c->d_table, c->table_stride, c->d_refcount);
        c->last_launches++;
    }
    if (c->timing) SPORK_CUDA(cudaEventRecord(c->t_ev[0], st));
    fork_clone_kernel<<<n, 256, 0, st>>>((const ForkDesc *)slot->d, c->d_free_list, c->d_table,
                                         c->table_stride, c->d_len, c->d_refcount,
                                         (uint8_t *)c->k_pool, (uint8_t *)c->v_pool, c->page_bytes,
                                         c->d_counters, (int)need, (int)(c->layer_k.size() * 2),
                                         (uint8_t *const *)c->d_layer_pools.p);
    c->last_launches++;
    if (c->timing) {
        SPORK_CUDA(cudaEventRecord(c->t_ev[1], st));
        SPORK_CUDA(cudaEventRecord(c->t_ev[2], st));
        c->t_valid = true;
    }
    SPORK_CUDA(cudaGetLastError());
    c->free_lb -= need;
    c->structure_epoch++;
    c->len_epoch++;
    return stage_done(c, slot, st);
}

static int drop_common(spork_ctx *c, int n, const int32_t *seq_ids, const int32_t *new_len,
                       cudaStream_t st) {
    // new_len == nullptr: release.  Errors are reported for the first offending request in array
    // order; a possibly-shared kept tail page BEFORE that request is resolved on the device first.
    if (c->mirror_stale) return SPORK_ERR_STALE;
    for (int i = 0; i < n; ++i) {
        int s = seq_ids[i];
        if (s >= 0 && s < c->cfg.max_seqs) c->h_scratch[s] = 0;
    }
    int n_ok = n, host_err = SPORK_OK;
    for (int i = 0; i < n; ++i) {
        int s = seq_ids[i];
        if (s < 0 || s >= c->cfg.max_seqs || !c->h_live[s] || c->h_scratch[s]++) {
            host_err = SPORK_ERR_INVALID_SEQ;
            n_ok = i;
            break;
        }
        if (new_len && (new_len[i] < 0 || new_len[i] > c->h_len[s])) {
            host_err = SPORK_ERR_INVALID;
            n_ok = i;
            break;
        }
    }
    if (n_ok == 0) return host_err;
    StageSlot *slot;
    int rc = stage_acquire(c, sizeof(DropDesc) * (size_t)n_ok, &slot);
    if (rc != SPORK_OK) return rc;
    DropDesc *d = (DropDesc *)slot->h;
    bool need_check = false;
    for (int i = 0; i < n_ok; ++i) {
        int s = seq_ids[i];
        d[i].seq = s;
        d[i].n_pages = pages_of(c->h_len[s]);
        d[i].new_len = new_len ? new_len[i] : 0;
        d[i].keep_pages = new_len ? pages_of(new_len[i]) : 0;
        d[i].agg_upto = 0;
        d[i].agg_mult = 1;
        // a partially filled kept tail page can only be shared below h_shared_upto
        if (new_len && (new_len[i] % PS) && new_len[i] / PS < c->h_shared_upto[s]) need_check = true;
    }
    if (host_err != SPORK_OK && !need_check) return host_err;
    if (!new_len && n_ok > 1) {
        // families: released children that still carry the same fork key (parent slot + fork call)
        std::unordered_map<uint64_t, int> leader;     // key -> index of the family's first member
        leader.reserve((size_t)n_ok);
        for (int i = 0; i < n_ok; ++i) {
            const int s = seq_ids[i];
            const uint64_t key = c->h_fork_key[s];
            const int nf = std::min(c->h_fork_nf[s], d[i].n_pages);
            if (key == 0 || nf == 0) continue;
            auto it = leader.find(key);
            if (it == leader.end()) {
                leader.emplace(key, i);
                d[i].agg_upto = nf;
                d[i].agg_mult = 1;
            } else {
                d[it->second].agg_mult++;
                d[i].agg_upto = nf;
                d[i].agg_mult = 0;
            }
        }
    }
    rc = stage_commit(c, slot, sizeof(DropDesc) * (size_t)n_ok, st);
    if (rc != SPORK_OK) return rc;
    if (need_check) {
        // exact answer needs the device refcounts: check, then read the flag (documented sync)
        SPORK_CUDA(cudaMemsetAsync(c->d_counters + 2, 0, 4, st));
        check_shared_kernel<<<ceil_div(n_ok, 256), 256, 0, st>>>((const DropDesc *)slot->d, n_ok,
                                                                 c->d_table, c->table_stride,
                                                                 c->d_refcount, c->d_counters + 2);
        c->last_launches++;
        int32_t flag = 0;
        SPORK_CUDA(cudaMemcpyAsync(&flag, c->d_counters + 2, 4, cudaMemcpyDeviceToHost, st));
        SPORK_CUDA(cudaStreamSynchronize(st));
        if (flag || host_err != SPORK_OK) {
            stage_done(c, slot, st);
            return flag ? SPORK_ERR_SHARED : host_err;
        }
    }
    c->fl_valid = false;        // pages are freed: the cached free list is no longer the lowest ids
    drop_pages_kernel<<<n, 256, 0, st>>>((const DropDesc *)slot->d, c->d_table, c->table_stride,
                                         c->d_len, c->d_refcount, c->d_counters);
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    for (int i = 0; i < n; ++i) {
        int s = seq_ids[i];
        if (new_len) {
            c->h_len[s] = new_len[i];
            c->h_shared_upto[s] = std::min(c->h_shared_upto[s], pages_of(new_len[i]));
            c->h_fork_key[s] = 0;      // a rolled-back sequence no longer mirrors its siblings
            lineage_truncate(c, s, pages_of(new_len[i]));
        } else {
            c->h_len[s] = 0;
            c->h_live[s] = 0;
            c->h_shared_upto[s] = 0;
            c->h_fork_key[s] = 0;
            lineage_reset(c, s);
        }
    }
    if (!new_len) c->n_live -= n;
    c->structure_epoch++;
    c->len_epoch++;
    return stage_done(c, slot, st);
}

extern "C" int spork_release(spork_ctx *c, int n, const int32_t *seq_ids, void *stream) {
    if (!c || n < 0 || (n > 0 && !seq_ids)) return SPORK_ERR_INVALID;
    c->last_launches = 0;
    if (n == 0) return SPORK_OK;
    return drop_common(c, n, seq_ids, nullptr, (cudaStream_t)stream);
}

extern "C" int spork_truncate(spork_ctx *c, int n, const int32_t *seq_ids, const int32_t *new_len,
                              void *stream) {
    if (!c || n < 0 || (n > 0 && (!seq_ids || !new_len))) return SPORK_ERR_INVALID;
    c->last_launches = 0;
    if (n == 0) return SPORK_OK;
    return drop_common(c, n, seq_ids, new_len, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------
// partial-token accept
// ---------------------------------------------------------------------------
namespace {

// one warp per sequence: index of the first draft position whose token differs from the target's
__global__ void __launch_bounds__(128) accept_len_kernel(const int32_t *__restrict__ q_indptr,
                                                         const int32_t *__restrict__ draft,
                                                         const int32_t *__restrict__ target, int n,
                                                         int32_t *__restrict__ accept_len) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n) return;
    const int b = q_indptr[w], e = q_indptr[w + 1];
    int first = e - b;
    for (int j0 = b; j0 < e; j0 += 32) {
        const int j = j0 + lane;
        const bool mismatch = j < e && draft[j] != target[j];
        const unsigned m = __ballot_sync(0xffffffffu, mismatch);
        if (m) {
            first = j0 - b + __ffs(m) - 1;
            break;
        }
    }
    if (lane == 0) accept_len[w] = first;
}

}  // namespace

extern "C" int spork_accept(spork_ctx *c, int n, const int32_t *seq_ids, const int32_t *q_indptr,
                            const int32_t *draft_tokens, const int32_t *target_tokens,
                            int32_t *accept_len_out, void *stream) {
    if (!c || n < 0) return SPORK_ERR_INVALID;
    c->last_launches = 0;
    if (n == 0) return SPORK_OK;
    if (!seq_ids || !q_indptr || !draft_tokens || !target_tokens || !accept_len_out || q_indptr[0] != 0)
        return SPORK_ERR_INVALID;
    if (c->mirror_stale) return SPORK_ERR_STALE;
    cudaStream_t st = (cudaStream_t)stream;
    for (int i = 0; i < n; ++i) {
        const int s = seq_ids[i], k = q_indptr[i + 1] - q_indptr[i];
        if (s < 0 || s >= c->cfg.max_seqs || !c->h_live[s]) return SPORK_ERR_INVALID_SEQ;
        if (k < 1 || k > c->h_len[s]) return SPORK_ERR_INVALID;
    }
    // q_indptr -> device, accept lengths <- device through one staging slot (the host needs the
    // lengths to mirror len[] anyway: this is the call's one documented synchronisation)
    const size_t ib = 4 * (size_t)(n + 1), ob = 4 * (size_t)n;
    StageSlot *slot;
    int rc = stage_acquire(c, ib + ob, &slot);
    if (rc != SPORK_OK) return rc;
    memcpy(slot->h, q_indptr, ib);
    rc = stage_commit(c, slot, ib, st);
    if (rc != SPORK_OK) return rc;
    int32_t *d_out = (int32_t *)((char *)slot->d + ib);
    accept_len_kernel<<<ceil_div(n, 4), 128, 0, st>>>((const int32_t *)slot->d, draft_tokens, target_tokens, n,
                                                      d_out);
    SPORK_CUDA(cudaGetLastError());
    SPORK_CUDA(cudaMemcpyAsync(accept_len_out, d_out, ob, cudaMemcpyDeviceToHost, st));
    SPORK_CUDA(cudaStreamSynchronize(st));
    rc = stage_done(c, slot, st);
    if (rc != SPORK_OK) return rc;
    std::vector<int32_t> new_len(n);
    for (int i = 0; i < n; ++i) {
        const int k = q_indptr[i + 1] - q_indptr[i];
        if (accept_len_out[i] < 0 || accept_len_out[i] > k) return SPORK_ERR_CUDA;
        new_len[i] = c->h_len[seq_ids[i]] - (k - accept_len_out[i]);
    }
    rc = drop_common(c, n, seq_ids, new_len.data(), st);
    c->last_launches++;     // + accept_len_kernel
    return rc;
}
