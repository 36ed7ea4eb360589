// libspork: attention planner.
//
// Per fork group the DEVICE block tables decide how many leading pages all
// members share (equal page id <=> same physical page); the host turns that and
// its mirrored lengths into a split-KV work list:
//   prefix segment  (one per group):  all members' rows x the shared pages, read once
//   suffix segment  (one per member): that member's rows x its private tokens
// Each segment is cut into equal chunks of whole 64-token tiles; one work item
// per (chunk, kv head, row block).  Segments with >= umma_min_rows rows (default: all) go
// to the tcgen05 kernel: in row blocks of <= 128 (one softmax pipe per CTA), or, when a
// segment has more than 128 rows (a verify call's drafts x group x GQA heads), in row
// blocks of <= 256 to the two-pipe variant, which fetches each K/V tile once for both
// halves.  The others go to the mma.sync kernel in row blocks of <= 64.
// Each kernel's items are sorted longest first and statically scheduled onto its
// persistent CTAs.
#include <limits.h>
#include <string.h>

#include <algorithm>
#include <functional>
#include <queue>
#include <utility>

#include "spork_internal.h"

using namespace spork;

namespace {

struct GroupDesc {
    int32_t begin, end, limit_pages, pad;
};

// one block per group: index of the first page at which the members' tables differ
__global__ void __launch_bounds__(256) lcp_kernel(const GroupDesc *__restrict__ groups,
                                                  const int32_t *__restrict__ seq_ids,
                                                  const int32_t *__restrict__ table, int table_stride,
                                                  int32_t *__restrict__ shared_out) {
    __shared__ int s_min;
    GroupDesc g = groups[blockIdx.x];
    if (threadIdx.x == 0) s_min = g.limit_pages;
    __syncthreads();
    const int32_t *row0 = table + (size_t)seq_ids[g.begin] * table_stride;
    for (int j = threadIdx.x; j < g.limit_pages; j += blockDim.x) {
        int v = row0[j];
        bool same = v >= 0;
        for (int m = g.begin + 1; m < g.end; ++m)
            same = same && table[(size_t)seq_ids[m] * table_stride + j] == v;
        if (!same) atomicMin(&s_min, j);
    }
    __syncthreads();
    if (threadIdx.x == 0) shared_out[blockIdx.x] = s_min;
}

constexpr int TILE_TOKENS = 64;
constexpr int MIN_CHUNK_TILES = 4;
constexpr int ROW_BLOCK = 64;
constexpr int ROW_BLOCK_UMMA = 128;
constexpr float ITEM_FIXED_COST = 1.5f;        // per-item overhead in 64-token-tile times
constexpr float ITEM_FIXED_COST_UMMA = 4.f;    // ... of the tcgen05 kernel (32 KiB of Q, 64 KiB of partials)
// ... of a tcgen05 item in the chunked schedule, which serves the many-row (compute-heavy) verify
// plans (sweep of the chunk length on config 4, k = 16: 630 / 587 / 650 / 669 us at 1 / 2 / 3 / 4 splits)
constexpr float ITEM_FIXED_COST_UMMA_CHUNKED = 8.f;

struct Segment {
    int table_seq, tok0, tok1;  // token range
    int qrow0, nq;              // q rows [qrow0, qrow0 + nq)
    int lim0;
    int part_base, nsplit, chunk_tiles;
    bool prefix;
    int kind;                   // 0: mma.sync / simt, 1: tcgen05 one pipe, 2: tcgen05 two pipes
    int row_block;
};

// longest first, then longest-processing-time-first onto `grid` persistent CTAs;
// cost of an item = its 64-token tiles (the bytes it streams) + 1 (fixed per-item work)
void schedule(std::vector<WorkItem> &items, int grid, std::vector<int32_t> &cta_ptr) {
    std::stable_sort(items.begin(), items.end(), [](const WorkItem &a, const WorkItem &b) {
        return (a.tok1 - a.tok0) > (b.tok1 - b.tok0);
    });
    cta_ptr.assign(grid + 1, 0);
    if (grid == 0) return;
    std::vector<int32_t> owner(items.size());
    std::priority_queue<std::pair<int64_t, int>, std::vector<std::pair<int64_t, int>>,
                        std::greater<std::pair<int64_t, int>>> heap;
    for (int b = 0; b < grid; ++b) heap.push({0, b});
    for (size_t i = 0; i < items.size(); ++i) {
        auto top = heap.top();
        heap.pop();
        owner[i] = top.second;
        cta_ptr[top.second + 1]++;
        top.first += 2 * ceil_div(items[i].tok1 - items[i].tok0, TILE_TOKENS) + 3;   // 2 x (tiles + 1.5)
        heap.push(top);
    }
    for (int b = 0; b < grid; ++b) cta_ptr[b + 1] += cta_ptr[b];
    std::vector<int32_t> fill(cta_ptr.begin(), cta_ptr.end() - 1);
    std::vector<WorkItem> sched(items.size());
    for (size_t i = 0; i < items.size(); ++i) sched[fill[owner[i]]++] = items[i];
    items.swap(sched);
}

}  // namespace

namespace spork {

int build_plan(spork_ctx *c, int n_groups, const int32_t *group_indptr, const int32_t *seq_ids,
               const int32_t *q_indptr, cudaStream_t st) {
    Plan &P = c->plan;
    if (n_groups < 0 || !group_indptr || group_indptr[0] != 0) return SPORK_ERR_INVALID;
    for (int g = 0; g < n_groups; ++g)
        if (group_indptr[g + 1] <= group_indptr[g]) return SPORK_ERR_INVALID;  // empty group
    const int n_seq = group_indptr[n_groups];
    if (n_seq > 0 && !seq_ids) return SPORK_ERR_INVALID;
    const bool verify = q_indptr != nullptr;
    for (int i = 0; i < n_seq; ++i) {
        int s = seq_ids[i];
        if (s < 0 || s >= c->cfg.max_seqs || !c->h_live[s]) return SPORK_ERR_INVALID_SEQ;
    }
    if (verify) {
        if (q_indptr[0] != 0) return SPORK_ERR_INVALID;
        for (int i = 0; i < n_seq; ++i) {
            int k = q_indptr[i + 1] - q_indptr[i];
            if (k < 1 || k > c->h_len[seq_ids[i]]) return SPORK_ERR_INVALID;
        }
    }
    const int n_qrows = verify ? q_indptr[n_seq] : n_seq;

    auto same = [](const std::vector<int32_t> &v, const int32_t *p, size_t n) {
        return v.size() == n && (n == 0 || memcmp(v.data(), p, n * 4) == 0);
    };
    // ---- level-2 cache: nothing changed since the last call -----------------
    if (P.valid && P.verify == verify && P.len_epoch == c->len_epoch &&
        P.structure_epoch == c->structure_epoch && same(P.group_indptr, group_indptr, n_groups + 1) &&
        same(P.seq_ids, seq_ids, n_seq) && (!verify || same(P.q_indptr, q_indptr, n_seq + 1))) {
        P.info.plan_cached = 1;
        return SPORK_OK;
    }
    P.valid = false;

    // ---- level-1 cache: shared page counts change only with fork / release / truncate ----
    if (!(P.shared_valid && P.shared_epoch == c->structure_epoch &&
          same(P.shared_key_indptr, group_indptr, n_groups + 1) &&
          same(P.shared_key_ids, seq_ids, n_seq))) {
        P.shared_pages.assign(n_groups, 0);
        bool any = false;
        for (int g = 0; g < n_groups; ++g) any = any || group_indptr[g + 1] - group_indptr[g] > 1;
        if (any) {
            size_t bytes = sizeof(GroupDesc) * (size_t)n_groups + 4 * (size_t)n_seq + 4 * (size_t)n_groups;
            StageSlot *slot;
            int rc = stage_acquire(c, bytes, &slot);
            if (rc != SPORK_OK) return rc;
            GroupDesc *gd = (GroupDesc *)slot->h;
            int32_t *ids = (int32_t *)(gd + n_groups);
            for (int g = 0; g < n_groups; ++g) {
                int lim = INT_MAX;
                for (int i = group_indptr[g]; i < group_indptr[g + 1]; ++i)
                    lim = std::min(lim, c->h_len[seq_ids[i]] / PS);
                if (group_indptr[g + 1] - group_indptr[g] < 2) lim = 0;
                gd[g] = {group_indptr[g], group_indptr[g + 1], lim, 0};
            }
            memcpy(ids, seq_ids, 4 * (size_t)n_seq);
            rc = stage_commit(c, slot, bytes - 4 * (size_t)n_groups, st);
            if (rc != SPORK_OK) return rc;
            int32_t *d_out = (int32_t *)((char *)slot->d + bytes - 4 * (size_t)n_groups);
            lcp_kernel<<<n_groups, 256, 0, st>>>((const GroupDesc *)slot->d,
                                                 (const int32_t *)((GroupDesc *)slot->d + n_groups),
                                                 c->d_table, c->table_stride, d_out);
            c->last_launches++;
            // documented sync: read back the per-group shared page counts
            SPORK_CUDA(cudaMemcpyAsync(P.shared_pages.data(), d_out, 4 * (size_t)n_groups,
                                       cudaMemcpyDeviceToHost, st));
            SPORK_CUDA(cudaStreamSynchronize(st));
        }
        P.shared_valid = true;
        P.shared_epoch = c->structure_epoch;
        P.shared_key_indptr.assign(group_indptr, group_indptr + n_groups + 1);
        P.shared_key_ids.assign(seq_ids, seq_ids + n_seq);
    }

    // ---- segments ------------------------------------------------------------
    const int Hq = c->cfg.num_q_heads, Hkv = c->cfg.num_kv_heads, G = c->G;
    std::vector<Segment> segs;
    segs.reserve(n_groups + n_seq);
    std::vector<QRowDesc> qd(n_qrows);
    int64_t unique_tokens = 0, naive_tokens = 0;
    for (int g = 0; g < n_groups; ++g) {
        const int b = group_indptr[g], e = group_indptr[g + 1];
        int S = P.shared_pages[g] * PS;
        for (int i = b; i < e; ++i) {
            int L = c->h_len[seq_ids[i]];
            int k = verify ? q_indptr[i + 1] - q_indptr[i] : (L > 0 ? 1 : 0);
            S = std::min(S, ((L - k) / PS) * PS);
            naive_tokens += L;
        }
        if (e - b < 2 || S < 0) S = 0;
        const int gq0 = verify ? q_indptr[b] : b;
        const int gnq = (verify ? q_indptr[e] : e) - gq0;
        int pre_seg = -1;
        if (S > 0) {
            pre_seg = (int)segs.size();
            segs.push_back({seq_ids[b], 0, S, gq0, gnq, INT_MAX / 2, 0, 0, 0, true, 0, ROW_BLOCK});
        }
        unique_tokens += S;
        for (int i = b; i < e; ++i) {
            int L = c->h_len[seq_ids[i]];
            int q0 = verify ? q_indptr[i] : i;
            int k = verify ? q_indptr[i + 1] - q_indptr[i] : 1;
            int suf_seg = -1;
            if (L > S) {
                suf_seg = (int)segs.size();
                segs.push_back({seq_ids[i], S, L, q0, k, L - k, 0, 0, 0, false, 0, ROW_BLOCK});
            }
            unique_tokens += L - S;
            for (int j = 0; j < k; ++j) {
                QRowDesc &d = qd[q0 + j];
                d.pre_stream = pre_seg;  // segment index for now; stream = segment * Hkv (+ kv head)
                d.pre_off = (q0 + j - gq0) * G;
                d.suf_stream = suf_seg;
                d.suf_off = j * G;
            }
        }
    }

    // ---- chunking --------------------------------------------------------------
    const bool mma = c->cfg.dtype == SPORK_BF16 && c->cfg.head_dim == 128;
    const int grid_cap = mma ? attn_mma_grid(c) : c->num_sms * 4;
    int64_t total_cost = 0;
    for (Segment &s : segs) {
        const int rows = s.nq * G;
        s.kind = !(mma && rows >= c->umma_min_rows) ? 0 : (rows > ROW_BLOCK_UMMA && c->many_row_variant ? 2 : 1);
        s.row_block = s.kind == 0 ? ROW_BLOCK : (s.kind == 2 && c->many_row_variant == 1 ? 2 : 1) * ROW_BLOCK_UMMA;
        int tiles = ceil_div(s.tok1 - s.tok0, TILE_TOKENS);
        total_cost += (int64_t)tiles * Hkv * ceil_div(s.nq * G, s.row_block);
    }
    // ---- split-KV chunk length: the candidate that minimises the estimated step time --------
    // Unit = the time one CTA needs to stream a 64-token tile when every CTA is busy.  An item
    // costs its tiles plus a fixed part (Q staging, partial write-back); the partials are written
    // once and read once by the merge kernel, which all CTAs share.  Fewer, longer items cost less
    // overhead and less partial traffic; more, shorter items balance the persistent CTAs better.
    const int grid_cap_umma = mma ? attn_umma_grid(c, 0) : 0;
    const int grid_cap_umma2 = mma ? attn_umma_grid(c, c->many_row_variant) : 0;
    auto split = [&](int chunk_tiles, int64_t *part_rows_out, size_t *n_items_out) -> bool {
        int64_t part_rows = 0;
        size_t n_items = 0;
        for (Segment &s : segs) {
            int tiles = ceil_div(s.tok1 - s.tok0, TILE_TOKENS);
            s.nsplit = ceil_div(tiles, chunk_tiles);
            s.chunk_tiles = ceil_div(tiles, s.nsplit);
            s.nsplit = ceil_div(tiles, s.chunk_tiles);
            if (part_rows + (int64_t)s.nsplit * s.nq * Hq > INT_MAX) return false;
            s.part_base = (int)part_rows;
            part_rows += (int64_t)s.nsplit * s.nq * Hq;
            n_items += (size_t)s.nsplit * Hkv * ceil_div(s.nq * G, s.row_block);
        }
        *part_rows_out = part_rows;
        *n_items_out = n_items;
        return true;
    };
    auto makespan = [&](int kind, int grid) -> double {
        std::vector<float> cost;
        for (const Segment &s : segs) {
            if (s.kind != kind) continue;
            const int tiles = ceil_div(s.tok1 - s.tok0, TILE_TOKENS);
            const int n_rb = ceil_div(s.nq * G, s.row_block);
            for (int sp = 0; sp < s.nsplit; ++sp) {
                // a two-pipe CTA has the SM to itself: a tile takes it half the time of a one-pipe CTA
                const float t = ((float)std::min(s.chunk_tiles, tiles - sp * s.chunk_tiles) +
                                 (kind ? ITEM_FIXED_COST_UMMA_CHUNKED : ITEM_FIXED_COST)) *
                                (kind == 2 && c->many_row_variant == 1 ? 0.5f : 1.f);
                cost.insert(cost.end(), (size_t)Hkv * n_rb, t);
            }
        }
        if (cost.empty()) return 0.0;
        std::sort(cost.begin(), cost.end(), std::greater<float>());
        const int g = (int)std::min<size_t>(cost.size(), (size_t)grid);
        std::priority_queue<double, std::vector<double>, std::greater<double>> heap;
        for (int b = 0; b < g; ++b) heap.push(0.0);
        double mk = 0.0;
        for (float t : cost) {
            double v = heap.top() + t;
            heap.pop();
            heap.push(v);
            mk = std::max(mk, v);
        }
        return mk;
    };
    int chunk_tiles = MIN_CHUNK_TILES;
    int64_t part_rows = 0;
    size_t n_items = 0;
    {
        static const float mult[] = {1.f, 1.5f, 2.f, 3.f, 4.f, 6.f};
        bool heavy = false;      // some tcgen05 segment has several row blocks
        for (const Segment &sg : segs) heavy = heavy || (sg.kind != 0 && sg.nq * G > sg.row_block);
        double best = -1.0;
        int best_chunk = -1;
        const int row_bytes = c->cfg.head_dim * 4 + 4;
        const double tile_bytes = 2.0 * TILE_TOKENS * c->cfg.head_dim * c->elt;
        for (float m : mult) {
            const int64_t target = (int64_t)(grid_cap * m);
            const int ct = (int)std::max<int64_t>(MIN_CHUNK_TILES, (total_cost + target - 1) / target);
            if (ct == best_chunk) continue;
            int64_t pr;
            size_t ni;
            if (!split(ct, &pr, &ni)) continue;
            const double partial = 2.0 * (double)pr * row_bytes / tile_bytes / grid_cap;
            double est = makespan(0, grid_cap) + makespan(1, grid_cap_umma) + makespan(2, grid_cap_umma2) + partial;
            // Many-row verify plans are bound by the SMs, not by HBM: two co-resident CTAs speed each
            // other up when one runs dry, which the per-CTA makespan does not see.  Measured on
            // config 4 (k = 8, 16; sweep in DESIGN.md): 4.5 to 6 items per CTA is the sweet spot, so
            // candidates outside it are handicapped.
            if (heavy && (2 * ni < 9 * (size_t)grid_cap_umma || ni > 6 * (size_t)grid_cap_umma)) est *= 1.25;
            if (best < 0.0 || est < best) {
                best = est;
                best_chunk = ct;
            }
        }
        if (best_chunk < 0) return SPORK_ERR_INVALID;
        chunk_tiles = best_chunk;
        if (!split(chunk_tiles, &part_rows, &n_items)) return SPORK_ERR_INVALID;
    }
    for (QRowDesc &d : qd) {
        if (d.pre_stream >= 0) d.pre_stream *= Hkv;
        if (d.suf_stream >= 0) d.suf_stream *= Hkv;
    }
    std::vector<StreamDesc> streams(segs.size() * (size_t)Hkv);   // stream of (segment s, kv head h) = s * Hkv + h

    std::vector<WorkItem> items, items_umma, items_umma2;
    std::vector<int32_t> cta_ptr, cta_ptr_umma, cta_ptr_umma2;
    int n_prefix_items = 0;
    auto make_item = [&](const Segment &s, int h, int rb, int t0, int t1, int part_base) {
        WorkItem it{};
        it.table_seq = s.table_seq;
        it.tok0 = t0;
        it.tok1 = t1;
        it.kvh = h;
        it.qrow0 = s.qrow0;
        it.rb0 = rb;
        it.nrows = std::min(s.row_block, s.nq * G - rb);
        it.lim0 = s.lim0;
        it.part_base = part_base;
        n_prefix_items += s.prefix;
        return it;
    };

    // ---- stream-K schedule: when every segment is ONE row block of the one-pipe tcgen05 kernel (all
    // decode plans, verify with few drafts), the segments are laid end to end, longest first, and cut
    // into contiguous runs of equal cost (tiles + a fixed cost per piece), one run per gang of Hkv CTAs:
    // every CTA streams the same number of bytes and a segment is split only where a gang boundary
    // falls (fewest partials).
    bool stream_k = mma && c->stream_k && !segs.empty();
    for (const Segment &s : segs) stream_k = stream_k && s.kind == 1 && s.nq * G <= s.row_block;
    if (stream_k) {
        // CTAs work in gangs of Hkv: a gang walks the same token run, CTA h of the gang on kv head h, so
        // the Hkv blocks of a page (contiguous in the pool) are fetched at the same time
        struct Str { int seg, tiles; };
        std::vector<Str> order;
        order.reserve(segs.size());
        int64_t tiles_total = 0;
        for (size_t si = 0; si < segs.size(); ++si) {
            const int tiles = ceil_div(segs[si].tok1 - segs[si].tok0, TILE_TOKENS);
            order.push_back({(int)si, tiles});
            tiles_total += tiles;
        }
        std::stable_sort(order.begin(), order.end(), [](const Str &a, const Str &b) { return a.tiles > b.tiles; });
        const int n_gangs = (int)std::min<int64_t>(std::max(1, grid_cap_umma / Hkv),
                                                  std::max<int64_t>(1, tiles_total / MIN_CHUNK_TILES));
        const int G_ = n_gangs * Hkv;
        const double c0 = ITEM_FIXED_COST_UMMA;
        const double budget = ((double)tiles_total + c0 * ((double)order.size() + n_gangs)) / n_gangs;
        std::vector<std::vector<WorkItem>> per_cta(G_);
        int gang = 0;
        double room = budget;            // cost the current gang can still take
        part_rows = 0;
        for (const Str &st_ : order) {
            const Segment &s = segs[st_.seg];
            const int rows = s.nq * G;
            if (part_rows > INT_MAX - (int64_t)rows * Hkv * (n_gangs + 1)) return SPORK_ERR_INVALID;
            const int seg_base = (int)part_rows;   // partial row of (split sp, head h, row i) = base + (sp * Hkv + h) * rows + i
            int nsplit = 0, done = 0;              // pieces so far, tiles of the segment already assigned
            while (done < st_.tiles) {
                const int left = st_.tiles - done;
                int take;
                if (gang == n_gangs - 1) {
                    take = left;         // the last gang takes what remains
                } else {
                    take = (int)std::min<double>(left, std::floor(room - c0));
                    if (take < std::min(left, MIN_CHUNK_TILES)) {   // no room for a useful piece: next gang
                        ++gang;
                        room = budget;
                        continue;
                    }
                    if (left - take > 0 && left - take < MIN_CHUNK_TILES) take = left;   // no crumbs
                }
                const int t0 = s.tok0 + done * TILE_TOKENS;
                const int t1 = std::min(s.tok1, t0 + take * TILE_TOKENS);
                for (int h = 0; h < Hkv; ++h)
                    per_cta[gang * Hkv + h].push_back(make_item(s, h, 0, t0, t1, seg_base + (nsplit * Hkv + h) * rows));
                nsplit++;
                done += take;
                room -= take + c0;
            }
            for (int h = 0; h < Hkv; ++h)
                streams[(size_t)st_.seg * Hkv + h] = StreamDesc{seg_base + h * rows, nsplit, Hkv * rows, 0};
            part_rows += (int64_t)nsplit * Hkv * rows;
        }
        cta_ptr_umma.assign(G_ + 1, 0);
        for (int b2 = 0; b2 < G_; ++b2) {
            cta_ptr_umma[b2 + 1] = cta_ptr_umma[b2] + (int)per_cta[b2].size();
            items_umma.insert(items_umma.end(), per_cta[b2].begin(), per_cta[b2].end());
        }
        chunk_tiles = (int)budget;
        cta_ptr.assign(1, 0);
        cta_ptr_umma2.assign(1, 0);
    } else {
        // ---- equal chunks per segment, items longest first, LPT onto each kernel's CTAs ----
        items.reserve(n_items);
        for (size_t si = 0; si < segs.size(); ++si) {
            const Segment &s = segs[si];
            const int rows = s.nq * G;
            for (int h = 0; h < Hkv; ++h)
                streams[si * Hkv + h] = StreamDesc{s.part_base + h * rows, s.nsplit, s.nq * Hq, 0};
            std::vector<WorkItem> &dst = s.kind == 2 ? items_umma2 : (s.kind == 1 ? items_umma : items);
            for (int sp = 0; sp < s.nsplit; ++sp) {
                int t0 = s.tok0 + sp * s.chunk_tiles * TILE_TOKENS;
                int t1 = std::min(s.tok1, t0 + s.chunk_tiles * TILE_TOKENS);
                for (int h = 0; h < Hkv; ++h)
                    for (int rb = 0; rb < rows; rb += s.row_block)
                        dst.push_back(make_item(s, h, rb, t0, t1, s.part_base + sp * s.nq * Hq + h * rows + rb));
            }
        }
        const int g0_ = (int)std::min<size_t>(items.size(), (size_t)grid_cap);
        if (mma) {
            schedule(items, g0_, cta_ptr);
            schedule(items_umma, (int)std::min<size_t>(items_umma.size(), (size_t)grid_cap_umma), cta_ptr_umma);
            schedule(items_umma2, (int)std::min<size_t>(items_umma2.size(), (size_t)grid_cap_umma2), cta_ptr_umma2);
        } else {
            std::stable_sort(items.begin(), items.end(), [](const WorkItem &a, const WorkItem &b) {
                return (a.tok1 - a.tok0) > (b.tok1 - b.tok0);
            });
            cta_ptr.assign(g0_ + 1, 0);
            cta_ptr_umma.assign(1, 0);
            cta_ptr_umma2.assign(1, 0);
        }
    }
    const int grid = (int)cta_ptr.size() - 1;
    const int grid_umma = (int)cta_ptr_umma.size() - 1;
    const int grid_umma2 = (int)cta_ptr_umma2.size() - 1;
    const int n_items_mma = (int)items.size();
    items.insert(items.end(), items_umma.begin(), items_umma.end());
    items.insert(items.end(), items_umma2.begin(), items_umma2.end());
    cta_ptr.insert(cta_ptr.end(), cta_ptr_umma.begin(), cta_ptr_umma.end());
    cta_ptr.insert(cta_ptr.end(), cta_ptr_umma2.begin(), cta_ptr_umma2.end());

    // ---- upload (the previous plan's buffers may still be in use by queued kernels) -----------
    if (c->plan_ev_pending) {
        SPORK_CUDA(cudaEventSynchronize(c->plan_ev));
        c->plan_ev_pending = false;
    }
    size_t ib = items.size() * sizeof(WorkItem), qb = qd.size() * sizeof(QRowDesc);
    const size_t cb = cta_ptr.size() * 4;
    int rc = devbuf_reserve(&P.items, ib + 64, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&P.qdesc, qb + 64, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&P.cta_ptr, cb + 64, st);
    const size_t sb = streams.size() * sizeof(StreamDesc);
    if (rc == SPORK_OK) rc = devbuf_reserve(&P.streams, sb + 64, st);

    if (rc == SPORK_OK) rc = devbuf_reserve(&c->ws_o, (size_t)part_rows * c->cfg.head_dim * 4 + 64, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&c->ws_lse, (size_t)part_rows * 4 + 64, st);
    if (rc != SPORK_OK) return rc;
    if (ib + qb) {
        StageSlot *slot;
        rc = stage_acquire(c, ib + qb + cb + sb, &slot);
        if (rc != SPORK_OK) return rc;
        if (ib) memcpy(slot->h, items.data(), ib);
        if (qb) memcpy((char *)slot->h + ib, qd.data(), qb);
        memcpy((char *)slot->h + ib + qb, cta_ptr.data(), cb);
        if (sb) memcpy((char *)slot->h + ib + qb + cb, streams.data(), sb);
        rc = stage_commit(c, slot, ib + qb + cb + sb, st);
        if (rc != SPORK_OK) return rc;
        if (ib) SPORK_CUDA(cudaMemcpyAsync(P.items.p, slot->d, ib, cudaMemcpyDeviceToDevice, st));
        if (qb)
            SPORK_CUDA(cudaMemcpyAsync(P.qdesc.p, (char *)slot->d + ib, qb, cudaMemcpyDeviceToDevice, st));
        SPORK_CUDA(cudaMemcpyAsync(P.cta_ptr.p, (char *)slot->d + ib + qb, cb, cudaMemcpyDeviceToDevice, st));
        if (sb)
            SPORK_CUDA(cudaMemcpyAsync(P.streams.p, (char *)slot->d + ib + qb + cb, sb, cudaMemcpyDeviceToDevice, st));
        rc = stage_done(c, slot, st);
        if (rc != SPORK_OK) return rc;
    }

    P.n_items = n_items_mma;
    P.n_items_umma = (int)items_umma.size();
    P.n_items_umma2 = (int)items_umma2.size();
    P.grid = grid;
    P.grid_umma = grid_umma;
    P.grid_umma2 = grid_umma2;
    P.variant2 = c->many_row_variant == 2 ? 2 : 1;
    P.n_qrows = n_qrows;
    P.verify = verify;
    P.len_epoch = c->len_epoch;
    P.structure_epoch = c->structure_epoch;
    P.group_indptr.assign(group_indptr, group_indptr + n_groups + 1);
    P.seq_ids.assign(seq_ids, seq_ids + n_seq);
    if (verify) P.q_indptr.assign(q_indptr, q_indptr + n_seq + 1); else P.q_indptr.clear();
    P.info = spork_plan_info{};
    P.info.n_items = P.n_items + P.n_items_umma + P.n_items_umma2;
    P.info.n_umma_items = P.n_items_umma + P.n_items_umma2;
    P.info.n_two_pipe_items = P.n_items_umma2;
    P.info.n_prefix_items = n_prefix_items;
    P.info.chunk_tokens = chunk_tiles * TILE_TOKENS;
    P.info.kernel = !mma ? 0 : (P.info.n_umma_items == 0 ? 1 : (P.n_items == 0 ? 2 : 3));
    P.info.plan_cached = 0;
    P.info.stream_k = stream_k ? 1 : 0;
    P.info.unique_tokens = unique_tokens;
    P.info.naive_tokens = naive_tokens;
    P.info.partial_rows = part_rows;
    P.valid = true;
    return SPORK_OK;
}

}  // namespace spork
