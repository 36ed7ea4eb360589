// libspork: attention planner (host).
//
// Per fork group the HOST lineage (which incarnation allocated each page of a sequence, kept up to
// date by append / fork / truncate / release) says which leading pages its members share; no device
// read-back is needed.  The group becomes a trie of cascade levels (Algorithm 1
// steps 4-6: probe r is forked after r * s further CoT tokens, so it shares
// P + r * s tokens with the main stream, not just P):
//   shared segment (one per trie node with >= 2 members): those members' rows x the pages they
//                   share beyond their parent node, read once
//   private tail   (one per member): that member's rows x its remaining tokens
// Each segment is cut into pieces of whole 64-token tiles; one work item per (piece, kv head, row
// block).  Segments with >= umma_min_rows rows (default: all) go to the tcgen05 kernel in row blocks
// of <= 128 (or <= 256 on the two-pipe variant), the others to the mma.sync kernel in row blocks of
// <= 64.  Items are statically scheduled onto each kernel's persistent CTAs.
//
// A plan does not bake in the lengths of the private tails: their last piece ends at the DEVICE
// length of its sequence (ITEM_LEN_TOK1), so a plan built once serves the decode loop
// {append one token to every stream; attend} (Alg. 1 step 5) until some sequence has
// grown by GROW_WINDOW tokens (one 64-token tile of imbalance) or the batch / the sharing changes.
#include <limits.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <functional>
#include <queue>
#include <utility>

#include "spork_internal.h"

using namespace spork;

// ---------------------------------------------------------------------------
// lineage
// ---------------------------------------------------------------------------
namespace spork {

void lineage_reset(spork_ctx *c, int s) {
    c->h_lin[s].n = 0;
    c->h_uid[s] = c->next_uid++;
}

static void lineage_push(Lineage &l, uint64_t uid, int end) {
    if (l.n > 0 && l.uid[l.n - 1] == uid) {
        l.end[l.n - 1] = end;
        return;
    }
    if (l.n == Lineage::MAX_RUNS) {
        // out of runs: the deepest run swallows what follows under the slot's own (fresh) label, which
        // nobody else holds -> sharing beyond this point is under-stated, never over-stated
        l.uid[l.n - 1] = uid;
        l.end[l.n - 1] = end;
        return;
    }
    l.uid[l.n] = uid;
    l.end[l.n] = end;
    l.n++;
}

void lineage_grow(spork_ctx *c, int s, int n_pages) {
    Lineage &l = c->h_lin[s];
    if (n_pages > l.pages()) lineage_push(l, c->h_uid[s], n_pages);
}

static void lineage_clip(Lineage &l, int keep) {
    while (l.n > 0 && (l.n > 1 ? l.end[l.n - 2] : 0) >= keep) l.n--;
    if (l.n > 0 && l.end[l.n - 1] > keep) l.end[l.n - 1] = keep;
}

void lineage_fork(spork_ctx *c, int child, int parent, int len) {
    const int nf = len / PS;
    c->h_lin[child] = c->h_lin[parent];
    lineage_clip(c->h_lin[child], nf);
    c->h_uid[child] = c->next_uid++;
    if (len % PS) lineage_push(c->h_lin[child], c->h_uid[child], nf + 1);   // the duplicated tail page
}

void lineage_truncate(spork_ctx *c, int s, int keep_pages) {
    lineage_clip(c->h_lin[s], keep_pages);
    // pages this slot allocates from now on are new pages, even at indices it has held before
    c->h_uid[s] = c->next_uid++;
}

int lineage_lcp(const Lineage &a, const Lineage &b) {
    int lcp = 0;
    for (int i = 0; i < a.n && i < b.n; ++i) {
        if (a.uid[i] != b.uid[i]) break;
        lcp = std::min(a.end[i], b.end[i]);
        if (a.end[i] != b.end[i]) break;
    }
    return lcp;
}

uint64_t lineage_label(const Lineage &a, int page) {
    for (int i = 0; i < a.n; ++i)
        if (page < a.end[i]) return a.uid[i];
    return 0;
}

}  // namespace spork

namespace {

constexpr int TILE_TOKENS = 64;
constexpr int MIN_CHUNK_TILES = 4;
constexpr int ROW_BLOCK = 64;
constexpr int ROW_BLOCK_UMMA = 128;
constexpr int GROW_WINDOW = 64;                // tokens a sequence may grow before its plan is rebuilt
constexpr int MIN_LEVEL_SAVING = 128;          // a deeper cascade level must save at least this many token reads
constexpr float ITEM_FIXED_COST = 1.5f;        // per-item overhead in 64-token-tile times
constexpr float ITEM_FIXED_COST_UMMA = 4.f;    // ... of the tcgen05 kernel (32 KiB of Q, 64 KiB of partials)
// ... of its FP8-KV variant, whose tile is shorter and whose Q staging (two e4m3 terms) is longer.  Sweep on the
// e4m3 configs (us per step at 2 / 4 / 6 / 8 / 12): config 5: 227 / 238 / 213 / 213 / 219, config 3: 241 / 192 /
// 193 / 195 / 203, config 2: 64 / 59 / 62 / 63 / 66.  (The same sweep on bf16: 3 and 4 within 1 %, 1 and 2 far off.)
constexpr float ITEM_FIXED_COST_UMMA_F8 = 6.f;
// ... of a tcgen05 item in the chunked schedule, which serves the many-row (compute-heavy) verify
// plans (sweep of the chunk length on config 4, k = 16: 630 / 587 / 650 / 669 us at 1 / 2 / 3 / 4 splits)
constexpr float ITEM_FIXED_COST_UMMA_CHUNKED = 8.f;

struct Segment {
    int table_seq, tok0, tok1;  // token range
    int qrow0, nq;              // q rows: [qrow0, qrow0 + nq), or rowmap[rowmap .. rowmap + nq) if rowmap >= 0
    int rowmap;
    int lim0, lim_k;            // visibility: t <= lim0 + (q index in the segment); private tails: lim0 = len - lim_k
    bool shared;                // a cascade level (several members), not a private tail
    bool open_end;              // private tail: tok1 follows the sequence's length
    int part_base, nsplit, chunk_tiles;
    int kind;                   // 0: mma.sync / simt, 1: tcgen05 one pipe, 2: tcgen05 two pipes
    int row_block;
};

struct Member {
    int seq, L, k, q0, vis_pages;   // vis_pages: leading pages every one of its rows sees entirely
};

struct GroupBuilder {
    const spork_ctx *c;
    const std::vector<Member> &mem;
    std::vector<Segment> &segs;
    std::vector<std::vector<std::pair<int, int>>> &refs;   // per q row: (segment, row offset)
    std::vector<int32_t> &rowmap;
    int G;
    int max_depth = 1;

    void tail(int m, int start_pages) {
        const Member &x = mem[m];
        if (x.L <= start_pages * PS || x.k == 0) return;
        const int seg = (int)segs.size();
        Segment s{};
        s.table_seq = x.seq;
        s.tok0 = start_pages * PS;
        s.tok1 = x.L;
        s.qrow0 = x.q0;
        s.nq = x.k;
        s.rowmap = -1;
        s.lim0 = x.k > 1 ? x.L - x.k : INT_MAX / 2;     // one row: it sees every token of the range
        s.lim_k = x.k;
        s.shared = false;
        s.open_end = true;
        segs.push_back(s);
        for (int j = 0; j < x.k; ++j) refs[x.q0 + j].push_back({seg, j * G});
    }

    // shared segment: the rows of all members of M x tokens [start_pages * 16, end_pages * 16)
    void shared(const std::vector<int> &M, int start_pages, int end_pages) {
        const int seg = (int)segs.size();
        Segment s{};
        s.table_seq = mem[M[0]].seq;
        s.tok0 = start_pages * PS;
        s.tok1 = end_pages * PS;
        s.lim0 = INT_MAX / 2;
        s.lim_k = 0;
        s.shared = true;
        s.open_end = false;
        s.nq = 0;
        bool contiguous = true;
        for (size_t i = 0; i < M.size(); ++i) {
            const Member &x = mem[M[i]];
            if (i > 0 && x.q0 != mem[M[i - 1]].q0 + mem[M[i - 1]].k) contiguous = false;
            s.nq += x.k;
        }
        s.qrow0 = mem[M[0]].q0;
        s.rowmap = -1;
        if (!contiguous) {
            s.rowmap = (int)rowmap.size();
            for (int m : M)
                for (int j = 0; j < mem[m].k; ++j) rowmap.push_back(mem[m].q0 + j);
        }
        segs.push_back(s);
        int off = 0;
        for (int m : M) {
            for (int j = 0; j < mem[m].k; ++j) refs[mem[m].q0 + j].push_back({seg, (off + j) * G});
            off += mem[m].k;
        }
    }

    // pages all members of M hold in common and all of their rows see entirely
    int common_pages(const std::vector<int> &M) const {
        const Lineage &l0 = c->h_lin[mem[M[0]].seq];
        int common = mem[M[0]].vis_pages;
        for (size_t i = 1; i < M.size(); ++i) {
            common = std::min(common, mem[M[i]].vis_pages);
            common = std::min(common, lineage_lcp(l0, c->h_lin[mem[M[i]].seq]));
        }
        return common;
    }

    // single-level cascade (max_levels = 1, the round-1 planner): one shared segment per group
    void single_level(const std::vector<int> &M) {
        int common = 0;
        if (M.size() > 1) {
            common = common_pages(M);
            if (common > 0) shared(M, 0, common);
        }
        for (int m : M) tail(m, common);
    }

    // Members M hold the same pages [0, known_pages); tokens below start_pages * 16 are covered by the
    // segments above (start_pages <= known_pages); `depth` = shared segments above.
    void node(const std::vector<int> &M, int start_pages, int known_pages, int depth, int max_levels) {
        if (M.size() == 1 || depth >= max_levels || depth + 2 > MAX_ROW_REFS) {   // keep room for the private tail
            for (int m : M) tail(m, start_pages);
            return;
        }
        const int common = std::max(common_pages(M), known_pages);
        // a deeper level must pay for its item overhead (else its tokens stay with the levels below it);
        // the root level is always taken
        const int64_t saving = (int64_t)(common - start_pages) * PS * ((int64_t)M.size() - 1);
        if (common > start_pages && (depth == 0 || saving >= MIN_LEVEL_SAVING)) {
            shared(M, start_pages, common);
            start_pages = common;
            depth += 1;
            max_depth = std::max(max_depth, depth);
        }
        // split by the page each member holds at index `common` (members that end there, or whose
        // rows do not all see that page, are on their own)
        std::vector<std::pair<uint64_t, int>> key;
        key.reserve(M.size());
        for (int m : M) {
            const Member &x = mem[m];
            const uint64_t lab = x.vis_pages > common ? lineage_label(c->h_lin[x.seq], common) : 0;
            key.push_back({lab, m});
        }
        std::vector<char> done(M.size(), 0);
        for (size_t i = 0; i < M.size(); ++i) {
            if (done[i]) continue;
            std::vector<int> sub{key[i].second};
            done[i] = 1;
            if (key[i].first != 0)
                for (size_t j = i + 1; j < M.size(); ++j)
                    if (!done[j] && key[j].first == key[i].first) {
                        sub.push_back(key[j].second);
                        done[j] = 1;
                    }
            if (sub.size() == M.size()) {
                // cannot happen with consistent lineages (equal labels at `common` would have made the
                // common run longer); never loop
                for (int m : sub) tail(m, start_pages);
                return;
            }
            node(sub, start_pages, common + (sub.size() > 1 ? 1 : 0), depth, max_levels);
        }
    }
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

inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

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
    // ---- plan cache: same batch, same sharing, and either nothing changed or every sequence has
    // only grown, by less than GROW_WINDOW tokens (the open-ended items follow the device lengths) ----
    if (P.valid && P.verify == verify && P.structure_epoch == c->structure_epoch &&
        same(P.group_indptr, group_indptr, n_groups + 1) && same(P.seq_ids, seq_ids, n_seq) &&
        (!verify || same(P.q_indptr, q_indptr, n_seq + 1))) {
        bool ok = true;
        int64_t grown = 0;
        if (P.len_epoch != c->len_epoch) {
            ok = P.growable;
            for (int i = 0; ok && i < n_seq; ++i) {
                const int d = c->h_len[seq_ids[i]] - P.base_len[i];
                ok = d >= 0 && d < GROW_WINDOW;
                grown += d;
            }
        }
        if (ok) {
            P.info.plan_cached = 1;
            P.info.unique_tokens = P.base_unique + grown;
            P.info.naive_tokens = P.base_naive + grown;
            return SPORK_OK;
        }
    }
    P.valid = false;
    const auto t_begin = std::chrono::steady_clock::now();

    // ---- segments: one cascade trie per group ----------------------------------------------
    const int Hq = c->cfg.num_q_heads, Hkv = c->cfg.num_kv_heads, G = c->G;
    std::vector<Segment> segs;
    segs.reserve(n_groups + n_seq);
    std::vector<std::vector<std::pair<int, int>>> row_refs(n_qrows);
    std::vector<int32_t> rowmap;
    std::vector<Member> mem;
    int64_t naive_tokens = 0;
    int n_levels = 1;
    bool growable = true;
    P.base_len.resize(n_seq);
    for (int g = 0; g < n_groups; ++g) {
        const int b = group_indptr[g], e = group_indptr[g + 1];
        mem.clear();
        for (int i = b; i < e; ++i) {
            const int L = c->h_len[seq_ids[i]];
            const int k = verify ? q_indptr[i + 1] - q_indptr[i] : (L > 0 ? 1 : 0);
            mem.push_back({seq_ids[i], L, k, verify ? q_indptr[i] : i, std::max(0, (L - std::max(k, 1)) / PS)});
            naive_tokens += L;
            P.base_len[i] = L;
            growable = growable && L > 0;
        }
        GroupBuilder gb{c, mem, segs, row_refs, rowmap, G};
        std::vector<int> all(mem.size());
        for (size_t i = 0; i < mem.size(); ++i) all[i] = (int)i;
        if (c->cascade_levels <= 1) gb.single_level(all);
        else gb.node(all, 0, 0, 0, c->cascade_levels);
        n_levels = std::max(n_levels, gb.max_depth);
    }
    int64_t unique_tokens = 0;
    for (const Segment &s : segs) unique_tokens += s.tok1 - s.tok0;

    // ---- chunking --------------------------------------------------------------
    const bool f8 = c->cfg.dtype == SPORK_E4M3;     // tcgen05 kernel only (one-pipe shape), no mma.sync alternative
    const bool mma = (c->cfg.dtype == SPORK_BF16 || f8) && c->cfg.head_dim == 128;
    const int grid_cap = mma ? attn_mma_grid(c) : c->num_sms * 4;
    // the generic (CUDA-core) kernel runs one warp per row and one CTA per item: short pieces and
    // row blocks of one warp each, so that even a tiny batch spreads over many SMs
    const int min_chunk_tiles = mma ? MIN_CHUNK_TILES : 1;
    int64_t total_cost = 0;
    for (Segment &s : segs) {
        const int rows = s.nq * G;
        s.kind = !(mma && (f8 || rows >= c->umma_min_rows)) ? 0
                 : (!f8 && rows > ROW_BLOCK_UMMA && c->many_row_variant ? 2 : 1);
        s.row_block = s.kind == 0 ? (mma ? ROW_BLOCK : 4)
                                  : (s.kind == 2 && c->many_row_variant == 1 ? 2 : 1) * ROW_BLOCK_UMMA;
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
    // ---- stream-K schedule: when every segment is ONE row block of the one-pipe tcgen05 kernel (all
    // decode plans, verify with few drafts), the segments are laid end to end, longest first, and cut
    // into contiguous runs of equal cost (tiles + a fixed cost per piece), one run per gang of Hkv CTAs:
    // every CTA streams the same number of bytes and a segment is split only where a gang boundary
    // falls (fewest partials).
    bool stream_k = mma && c->stream_k && !segs.empty();
    for (const Segment &s : segs) stream_k = stream_k && s.kind == 1 && s.nq * G <= s.row_block;

    int chunk_tiles = min_chunk_tiles;
    int64_t part_rows = 0;
    size_t n_items = 0;
    if (!stream_k) {
        static const float mult[] = {1.f, 1.5f, 2.f, 3.f, 4.f, 6.f};
        bool heavy = false;      // some tcgen05 segment has several row blocks
        for (const Segment &sg : segs) heavy = heavy || (sg.kind != 0 && sg.nq * G > sg.row_block);
        double best = -1.0;
        int best_chunk = -1;
        const int row_bytes = c->cfg.head_dim * 4 + 4;
        const double tile_bytes = 2.0 * TILE_TOKENS * c->cfg.head_dim * c->elt;
        for (float m : mult) {
            const int64_t target = (int64_t)(grid_cap * m);
            const int ct = (int)std::max<int64_t>(min_chunk_tiles, (total_cost + target - 1) / target);
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
    std::vector<StreamDesc> streams(segs.size() * (size_t)Hkv);   // stream of (segment s, kv head h) = s * Hkv + h

    std::vector<WorkItem> items, items_umma, items_umma2;
    std::vector<int32_t> cta_ptr, cta_ptr_umma, cta_ptr_umma2;
    int n_prefix_items = 0;
    // `last`: the piece that ends where the segment ends
    auto make_item = [&](const Segment &s, int h, int rb, int t0, int t1, int part_base, bool last) {
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
        it.flags = 0;
        if (s.open_end && growable) {
            if (s.lim_k > 1) it.flags |= ITEM_LEN_LIM;
            if (last) it.flags |= ITEM_LEN_TOK1;
        }
        it.lim_k = s.lim_k;
        it.rowmap = s.rowmap;
        n_prefix_items += s.shared;
        return it;
    };

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
        const double c0 = f8 ? ITEM_FIXED_COST_UMMA_F8 : ITEM_FIXED_COST_UMMA;
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
                    per_cta[gang * Hkv + h].push_back(
                        make_item(s, h, 0, t0, t1, seg_base + (nsplit * Hkv + h) * rows, done + take == st_.tiles));
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
                        dst.push_back(make_item(s, h, rb, t0, t1, s.part_base + sp * s.nq * Hq + h * rows + rb,
                                                sp == s.nsplit - 1));
            }
        }
        const int g0_ = (int)std::min<size_t>(items.size(), (size_t)grid_cap);
        if (mma) {
            schedule(items, g0_, cta_ptr);
            schedule(items_umma, (int)std::min<size_t>(items_umma.size(), (size_t)grid_cap_umma), cta_ptr_umma);
            schedule(items_umma2, (int)std::min<size_t>(items_umma2.size(), (size_t)grid_cap_umma2), cta_ptr_umma2);
        } else {
            // the generic kernel: one CTA per item
            std::stable_sort(items.begin(), items.end(), [](const WorkItem &a, const WorkItem &b) {
                return (a.tok1 - a.tok0) > (b.tok1 - b.tok0);
            });
            cta_ptr.assign(1, 0);
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

    // ---- merge descriptors ---------------------------------------------------------------------
    std::vector<QRowDesc> qd(n_qrows);
    std::vector<RowRef> refs;
    refs.reserve((size_t)n_qrows * 2);
    for (int r = 0; r < n_qrows; ++r) {
        qd[r].ref0 = (int)refs.size();
        qd[r].nref = (int)row_refs[r].size();
        for (const auto &pr : row_refs[r]) refs.push_back({pr.first * Hkv, pr.second});
    }

    // ---- upload: one pinned staging slot -> one device buffer, stream-ordered (the kernels of the
    // previous call that still read the old plan are ahead of this copy on the same stream) ----
    const size_t ib = items.size() * sizeof(WorkItem), qb = qd.size() * sizeof(QRowDesc);
    const size_t rb_ = refs.size() * sizeof(RowRef), sb = streams.size() * sizeof(StreamDesc);
    const size_t cb = cta_ptr.size() * 4, mb = rowmap.size() * 4;
    const size_t o_items = 0, o_qd = align16(o_items + ib), o_refs = align16(o_qd + qb), o_str = align16(o_refs + rb_);
    const size_t o_cta = align16(o_str + sb), o_map = align16(o_cta + cb), total = align16(o_map + mb) + 64;
    int rc = devbuf_reserve(&P.blob, total, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&c->ws_o, (size_t)part_rows * c->cfg.head_dim * 4 + 64, st);
    if (rc == SPORK_OK) rc = devbuf_reserve(&c->ws_lse, (size_t)part_rows * 4 + 64, st);
    if (rc != SPORK_OK) return rc;
    if (ib + qb) {
        StageSlot *slot;
        rc = stage_acquire(c, total, &slot);
        if (rc != SPORK_OK) return rc;
        char *h = (char *)slot->h;
        if (ib) memcpy(h + o_items, items.data(), ib);
        if (qb) memcpy(h + o_qd, qd.data(), qb);
        if (rb_) memcpy(h + o_refs, refs.data(), rb_);
        if (sb) memcpy(h + o_str, streams.data(), sb);
        memcpy(h + o_cta, cta_ptr.data(), cb);
        if (mb) memcpy(h + o_map, rowmap.data(), mb);
        SPORK_CUDA(cudaMemcpyAsync(P.blob.p, slot->h, total - 64, cudaMemcpyHostToDevice, st));
        rc = stage_done(c, slot, st);
        if (rc != SPORK_OK) return rc;
    }
    const char *d = (const char *)P.blob.p;
    P.d_items = (const WorkItem *)(d + o_items);
    P.d_qdesc = (const QRowDesc *)(d + o_qd);
    P.d_refs = (const RowRef *)(d + o_refs);
    P.d_streams = (const StreamDesc *)(d + o_str);
    P.d_cta_ptr = (const int32_t *)(d + o_cta);
    P.d_rowmap = (const int32_t *)(d + o_map);

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
    P.growable = growable;
    P.base_unique = unique_tokens;
    P.base_naive = naive_tokens;
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
    P.info.plan_host_us = std::chrono::duration<float, std::micro>(std::chrono::steady_clock::now() - t_begin).count();
    P.info.plan_builds = ++c->plan_builds;
    P.info.n_levels = n_levels;
    P.valid = true;
    return SPORK_OK;
}

}  // namespace spork
