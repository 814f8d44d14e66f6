// Mask descriptor -> query groups / key ranges -> ordered tile tasks (host, integers only).
//
// "The custom mask is represented as a set of query groups and their admissible key
// ranges ... The kernel launches tasks (g, i), where i is a query tile inside Q_g.  Each task streams only
// the key ranges in K_g."  Teacher forcing (Eq. 8) and block-causal masks become "a small
// number of full query-key rectangles"; dense attention is one group with one range.
#include <algorithm>
#include <cstring>
#include <new>

#include "internal.hpp"

namespace aj {

static thread_local std::string g_error;

void set_error(const std::string &msg) { g_error = msg; }
aj_status fail(aj_status st, const std::string &msg) {
    g_error = msg;
    return st;
}
const char *last_error_cstr() { return g_error.c_str(); }

// Block boundaries of one half: [0, C1, C1 + C, C1 + 2C, ...] (R6).
static aj_status block_bounds(const aj_mask_desc &m, std::vector<int64_t> &b) {
    if (m.frame_len <= 0 || m.num_frames <= 0 || m.chunk_frames <= 0 || m.first_chunk_frames < 0)
        return fail(AJ_ERR_INVALID_ARG, "mask: frame_len, num_frames, chunk_frames must be > 0");
    int64_t first = m.first_chunk_frames > 0 ? m.first_chunk_frames : m.chunk_frames;
    if (first > m.num_frames || (m.num_frames - first) % m.chunk_frames != 0)
        return fail(AJ_ERR_INVALID_ARG, "mask: num_frames is not first_chunk_frames + k * chunk_frames");
    b.clear();
    b.push_back(0);
    for (int64_t f = first; f <= m.num_frames; f += m.chunk_frames) b.push_back(f * m.frame_len);
    return AJ_OK;
}

static void push_group(Lowered &out, int64_t q0, int64_t q1, std::initializer_list<KeyRange> rs, int32_t q_tz = 0) {
    out.q_begin.push_back((int32_t)q0);
    out.q_end.push_back((int32_t)q1);
    out.q_tz.push_back(q_tz);
    for (const KeyRange &r : rs) {
        if (r.k_end <= r.k_begin) continue;
        // merge with the previous range of this group when they touch (and promise the same about their tangents)
        if ((int32_t)out.ranges.size() > out.range_offset.back() && out.ranges.back().k_end == r.k_begin && out.ranges.back().tz == r.tz)
            out.ranges.back().k_end = r.k_end;
        else
            out.ranges.push_back(r);
    }
    out.range_offset.push_back((int32_t)out.ranges.size());
}

aj_status lower_mask(const aj_problem &p, const aj_mask_desc &m, Lowered &out) {
    out = Lowered();
    out.range_offset.push_back(0);
    std::vector<int64_t> bb;
    const int32_t tzk = m.tangent_zero;
    if (tzk != AJ_TANGENT_DENSE && tzk != AJ_TANGENT_CLEAN_ZERO && tzk != AJ_TANGENT_NONE)
        return fail(AJ_ERR_INVALID_ARG, "mask: unknown tangent_zero");
    if (tzk == AJ_TANGENT_CLEAN_ZERO && m.kind != AJ_MASK_TEACHER_FORCING && m.kind != AJ_MASK_RANGES)
        return fail(AJ_ERR_INVALID_ARG, "mask: AJ_TANGENT_CLEAN_ZERO needs a teacher-forcing or ranges mask");
    const int32_t all0 = tzk == AJ_TANGENT_NONE ? 1 : 0;       // every tangent is zero
    const int32_t clean0 = tzk != AJ_TANGENT_DENSE ? 1 : 0;    // the clean half's tangents are zero
    switch (m.kind) {
    case AJ_MASK_FULL:
        push_group(out, 0, p.Nq, {KeyRange{0, p.Nk, all0}}, all0);
        break;
    case AJ_MASK_BLOCK_CAUSAL: {
        if (aj_status st = block_bounds(m, bb)) return st;
        if (p.Nq != bb.back() || p.Nk != bb.back())
            return fail(AJ_ERR_INVALID_ARG, "block-causal mask: Nq and Nk must equal num_frames * frame_len");
        for (size_t i = 0; i + 1 < bb.size(); ++i)  // block i sees blocks <= i
            push_group(out, bb[i], bb[i + 1], {KeyRange{0, (int32_t)bb[i + 1], all0}}, all0);
        break;
    }
    case AJ_MASK_TEACHER_FORCING: {
        if (aj_status st = block_bounds(m, bb)) return st;
        const int64_t half = bb.back();
        if (p.Nq != 2 * half || p.Nk != 2 * half)
            return fail(AJ_ERR_INVALID_ARG, "teacher-forcing mask: Nq and Nk must equal 2 * num_frames * frame_len");
        for (size_t i = 0; i + 1 < bb.size(); ++i)  // clean block i -> clean blocks <= i
            push_group(out, bb[i], bb[i + 1], {KeyRange{0, (int32_t)bb[i + 1], clean0}}, clean0);
        for (size_t i = 0; i + 1 < bb.size(); ++i)  // noisy block i -> clean blocks < i, noisy block i
            push_group(out, half + bb[i], half + bb[i + 1],
                       {KeyRange{0, (int32_t)bb[i], clean0}, KeyRange{(int32_t)(half + bb[i]), (int32_t)(half + bb[i + 1]), all0}}, all0);
        break;
    }
    case AJ_MASK_RANGES: {
        if (m.num_groups < 0 || (m.num_groups > 0 && (!m.q_begin || !m.q_end || !m.range_offset)))
            return fail(AJ_ERR_INVALID_ARG, "ranges mask: null group arrays");
        if (m.num_groups > 0 && m.range_offset[0] != 0)
            return fail(AJ_ERR_INVALID_ARG, "ranges mask: range_offset[0] must be 0");
        std::vector<std::pair<int32_t, int32_t>> rows;
        for (int g = 0; g < m.num_groups; ++g) {
            int32_t q0 = m.q_begin[g], q1 = m.q_end[g];
            if (q0 < 0 || q1 > p.Nq || q0 >= q1)
                return fail(AJ_ERR_INVALID_ARG, "ranges mask: query group outside [0, Nq) or empty");
            int32_t r0 = m.range_offset[g], r1 = m.range_offset[g + 1];
            if (r1 < r0) return fail(AJ_ERR_INVALID_ARG, "ranges mask: range_offset must be non-decreasing");
            if (r1 > r0 && (!m.k_begin || !m.k_end)) return fail(AJ_ERR_INVALID_ARG, "ranges mask: null range arrays");
            out.q_begin.push_back(q0);
            out.q_end.push_back(q1);
            out.q_tz.push_back(all0 || (tzk == AJ_TANGENT_CLEAN_ZERO && m.q_tangent_zero && m.q_tangent_zero[g]) ? 1 : 0);
            int32_t prev_end = 0;
            for (int r = r0; r < r1; ++r) {
                int32_t k0 = m.k_begin[r], k1 = m.k_end[r];
                if (k0 < 0 || k1 > p.Nk || k0 >= k1 || k0 < prev_end)
                    return fail(AJ_ERR_INVALID_ARG, "ranges mask: key ranges must be non-empty, sorted, disjoint, inside [0, Nk)");
                const int32_t tz = all0 || (tzk == AJ_TANGENT_CLEAN_ZERO && m.k_tangent_zero && m.k_tangent_zero[r]) ? 1 : 0;
                if (r > r0 && out.ranges.back().k_end == k0 && out.ranges.back().tz == tz) out.ranges.back().k_end = k1;
                else out.ranges.push_back(KeyRange{k0, k1, tz});
                prev_end = k1;
            }
            out.range_offset.push_back((int32_t)out.ranges.size());
            rows.emplace_back(q0, q1);
        }
        std::sort(rows.begin(), rows.end());
        for (size_t i = 1; i < rows.size(); ++i)
            if (rows[i].first < rows[i - 1].second)
                return fail(AJ_ERR_INVALID_ARG, "ranges mask: query groups overlap");
        // rows in no group become key-less groups so that every output row is written (O = 0, tO = 0, lse = -inf)
        int32_t next = 0;
        rows.emplace_back(p.Nq, p.Nq);
        for (const auto &qr : rows) {
            if (qr.first > next) push_group(out, next, qr.first, {}, 1);
            next = std::max(next, qr.second);
        }
        break;
    }
    default:
        return fail(AJ_ERR_INVALID_ARG, "mask: unknown kind");
    }
    out.pairs_per_head = 0;
    for (size_t g = 0; g < out.q_begin.size(); ++g) {
        const int64_t rows = out.q_end[g] - out.q_begin[g];
        for (int r = out.range_offset[g]; r < out.range_offset[g + 1]; ++r) {
            const int64_t pairs = rows * (int64_t)(out.ranges[r].k_end - out.ranges[r].k_begin);
            out.pairs_per_head += pairs;
            out.pair_class[!out.ranges[r].tz ? 2 : out.q_tz[g] ? 0 : 1] += pairs;
        }
    }
    return AJ_OK;
}

// The mask seen from the keys (for dK, dV of the primal backward): key groups = maximal key intervals seen by the same
// set of rows, each with the sorted, merged row ranges that see it.  In `out` the roles are swapped: q_* are key
// intervals and `ranges` are query-row ranges.  Keys no row sees become range-less groups (their dK, dV are 0).
void transpose_lowered(const aj_problem &p, const Lowered &low, Lowered &out) {
    out = Lowered();
    out.range_offset.push_back(0);
    const size_t ng = low.q_begin.size();
    std::vector<size_t> order(ng);
    for (size_t g = 0; g < ng; ++g) order[g] = g;
    std::sort(order.begin(), order.end(), [&](size_t a, size_t b) { return low.q_begin[a] < low.q_begin[b]; });
    std::vector<int32_t> cuts{0, p.Nk};
    for (const KeyRange &r : low.ranges) { cuts.push_back(r.k_begin); cuts.push_back(r.k_end); }
    std::sort(cuts.begin(), cuts.end());
    cuts.erase(std::unique(cuts.begin(), cuts.end()), cuts.end());
    std::vector<KeyRange> rows, prev;
    for (size_t c = 0; c + 1 < cuts.size(); ++c) {
        const int32_t a = cuts[c], b = cuts[c + 1];
        rows.clear();
        for (size_t i = 0; i < ng; ++i) {
            const size_t g = order[i];
            bool covered = false;
            for (int r = low.range_offset[g]; r < low.range_offset[g + 1] && !covered; ++r)
                covered = low.ranges[r].k_begin <= a && b <= low.ranges[r].k_end;
            if (!covered || low.q_end[g] <= low.q_begin[g]) continue;
            if (!rows.empty() && rows.back().k_end == low.q_begin[g]) rows.back().k_end = low.q_end[g];
            else rows.push_back(KeyRange{low.q_begin[g], low.q_end[g], 0});
        }
        bool same = !out.q_begin.empty() && out.q_end.back() == a && rows.size() == prev.size();
        for (size_t i = 0; same && i < rows.size(); ++i) same = rows[i].k_begin == prev[i].k_begin && rows[i].k_end == prev[i].k_end;
        if (same) { out.q_end.back() = b; continue; }       // same rows as the interval before: extend it
        out.q_begin.push_back(a);
        out.q_end.push_back(b);
        out.q_tz.push_back(0);
        out.ranges.insert(out.ranges.end(), rows.begin(), rows.end());
        out.range_offset.push_back((int32_t)out.ranges.size());
        prev = rows;
    }
    out.pairs_per_head = low.pairs_per_head;
    out.pair_class[2] = low.pairs_per_head;
}

static void order_tasks(std::vector<aj_task> &tasks) {
    // Longest-first so that the persistent CTAs finish together; ties keep (b, h, group/tile) order so that
    // tasks streaming the same keys of the same head run at the same time and share them in L2.
    std::stable_sort(tasks.begin(), tasks.end(),
                     [](const aj_task &x, const aj_task &y) { return x.num_kv_tiles > y.num_kv_tiles; });
}

void build_tasks(const aj_problem &p, const Lowered &low, int32_t tile_q, int32_t tile_k, Entries &ent,
                 std::vector<aj_task> &tasks) {
    tasks.clear();
    ent = Entries();
    for (const KeyRange &r : low.ranges) {
        ent.k_begin.push_back(r.k_begin); ent.k_end.push_back(r.k_end);
        ent.row_begin.push_back(0); ent.row_end.push_back(tile_q);
        ent.k_tz.push_back(r.tz);
    }
    for (int32_t b = 0; b < p.B; ++b)
        for (int32_t h = 0; h < p.H; ++h)
            for (size_t g = 0; g < low.q_begin.size(); ++g) {
                int32_t r0 = low.range_offset[g], r1 = low.range_offset[g + 1];
                int32_t kv_tiles = 0;
                bool primal = low.q_tz[g] != 0;
                for (int r = r0; r < r1; ++r) {
                    kv_tiles += (low.ranges[r].k_end - low.ranges[r].k_begin + tile_k - 1) / tile_k;
                    primal = primal && low.ranges[r].tz;
                }
                // query tiles start at the group start (R8); the last one may be partial
                for (int32_t q = low.q_begin[g]; q < low.q_end[g]; q += tile_q) {
                    aj_task t;
                    t.b = b; t.h = h; t.q_begin = q;
                    t.q_rows = std::min(tile_q, low.q_end[g] - q);
                    t.range_begin = r0; t.range_count = r1 - r0;
                    t.num_kv_tiles = kv_tiles; t.group = (int32_t)g;
                    t.flags = primal ? AJ_TASK_PRIMAL_ONLY : 0;
                    tasks.push_back(t);
                }
            }
    order_tasks(tasks);
}

void build_tasks_packed(const aj_problem &p, const Lowered &low, int32_t tile_q, int32_t tile_k, Entries &ent,
                        std::vector<aj_task> &tasks) {
    tasks.clear();
    ent = Entries();
    const size_t ng = low.q_begin.size();
    std::vector<size_t> order(ng);                     // groups in row order (they are disjoint)
    for (size_t g = 0; g < ng; ++g) order[g] = g;
    std::sort(order.begin(), order.end(), [&](size_t a, size_t b) { return low.q_begin[a] < low.q_begin[b]; });
    struct Run { int32_t lo, hi; };
    struct TileInfo { int32_t q_begin, q_rows, ent_begin, ent_count, kv_tiles, flags; };
    std::vector<TileInfo> tiles;
    size_t first = 0;                                  // first group (in row order) that may reach this tile
    std::vector<int32_t> cuts;
    std::vector<Run> runs, prev_runs;
    for (int32_t t0 = 0; t0 < p.Nq; t0 += tile_q) {
        const int32_t t1 = std::min(p.Nq, t0 + tile_q);
        while (first < ng && low.q_end[order[first]] <= t0) ++first;
        size_t last = first;                           // groups [first, last) intersect rows [t0, t1)
        while (last < ng && low.q_begin[order[last]] < t1) ++last;
        cuts.clear();
        for (size_t i = first; i < last; ++i) {
            const size_t g = order[i];
            for (int r = low.range_offset[g]; r < low.range_offset[g + 1]; ++r) {
                cuts.push_back(low.ranges[r].k_begin);
                cuts.push_back(low.ranges[r].k_end);
            }
        }
        std::sort(cuts.begin(), cuts.end());
        cuts.erase(std::unique(cuts.begin(), cuts.end()), cuts.end());
        TileInfo ti{t0, t1 - t0, (int32_t)ent.size(), 0, 0, 0};
        size_t open_begin = ent.size();                // entries of the key interval being extended
        prev_runs.clear();
        int32_t prev_end = -1, prev_tz = -1;
        bool primal = true;                            // tQ of every row and tK, tV of every key are structurally zero
        for (size_t i = first; i < last; ++i) primal = primal && low.q_tz[order[i]];
        for (size_t c = 0; c + 1 < cuts.size(); ++c) {
            const int32_t a = cuts[c], bnd = cuts[c + 1];
            // rows of the tile that see keys [a, bnd): union over the groups whose ranges cover it, as maximal runs
            runs.clear();
            int32_t tz = 1;                            // zero only if every covering range says so
            for (size_t i = first; i < last; ++i) {
                const size_t g = order[i];
                bool covered = false;
                for (int r = low.range_offset[g]; r < low.range_offset[g + 1] && !covered; ++r)
                    if ((covered = low.ranges[r].k_begin <= a && bnd <= low.ranges[r].k_end)) tz = tz && low.ranges[r].tz;
                if (!covered) continue;
                const int32_t lo = std::max(low.q_begin[g], t0) - t0, hi = std::min(low.q_end[g], t1) - t0;
                if (!runs.empty() && runs.back().hi == lo) runs.back().hi = hi;
                else runs.push_back(Run{lo, hi});
            }
            if (runs.empty()) { prev_runs.clear(); prev_end = -1; continue; }
            primal = primal && tz;
            bool same = prev_end == a && prev_tz == tz && runs.size() == prev_runs.size();
            for (size_t i = 0; same && i < runs.size(); ++i) same = runs[i].lo == prev_runs[i].lo && runs[i].hi == prev_runs[i].hi;
            if (same) {                                // same rows as the interval before and adjacent keys: extend
                for (size_t e = open_begin; e < ent.size(); ++e) ent.k_end[e] = bnd;
            } else {
                open_begin = ent.size();
                for (const Run &r : runs) {
                    ent.k_begin.push_back(a); ent.k_end.push_back(bnd);
                    ent.row_begin.push_back(r.lo); ent.row_end.push_back(r.hi);
                    ent.k_tz.push_back(tz);
                }
            }
            prev_runs = runs;
            prev_end = bnd;
            prev_tz = tz;
        }
        ti.flags = primal ? AJ_TASK_PRIMAL_ONLY : 0;
        ti.ent_count = (int32_t)ent.size() - ti.ent_begin;
        for (int32_t e = ti.ent_begin; e < ti.ent_begin + ti.ent_count; ++e)
            ti.kv_tiles += (ent.k_end[e] - ent.k_begin[e] + tile_k - 1) / tile_k;
        tiles.push_back(ti);
    }
    for (int32_t b = 0; b < p.B; ++b)
        for (int32_t h = 0; h < p.H; ++h)
            for (const TileInfo &ti : tiles) {
                aj_task t;
                t.b = b; t.h = h; t.q_begin = ti.q_begin; t.q_rows = ti.q_rows;
                t.range_begin = ti.ent_begin; t.range_count = ti.ent_count;
                t.num_kv_tiles = ti.kv_tiles; t.group = -1; t.flags = ti.flags;
                tasks.push_back(t);
            }
    order_tasks(tasks);
}

// Cost of a task on a CTA pair in units of a tenth of a full pair-step (two key tiles, all 6 contractions = 48 MMAs):
// a pair-step whose keys have zero tangents runs 32 MMAs, a primal-only one 16 (but is bound by the exponentials of
// its softmax, not by the MMAs); the constant covers the Q load and the epilogue.
static int64_t task_cost(const aj_task &t, const Entries &ent, int32_t tile_k) {
    constexpr int64_t W_FULL = 10, W_KEYZERO = 7, W_PRIMAL = 5, W_TASK = 10;
    const int64_t steps = (t.num_kv_tiles + 1) / 2;
    if (t.flags & AJ_TASK_PRIMAL_ONLY) return W_TASK + W_PRIMAL * steps;
    int64_t cost = W_TASK, tile = 0;
    bool step_tz = true;
    for (int32_t e = t.range_begin; e < t.range_begin + t.range_count; ++e) {
        const int64_t n = (ent.k_end[e] - ent.k_begin[e] + tile_k - 1) / tile_k;
        const bool tz = !ent.k_tz.empty() && ent.k_tz[e];
        for (int64_t i = 0; i < n; ++i, ++tile) {
            if ((tile & 1) == 0) step_tz = tz;
            else { step_tz = step_tz && tz; cost += step_tz ? W_KEYZERO : W_FULL; }
        }
    }
    if (tile & 1) cost += step_tz ? W_KEYZERO : W_FULL;
    return cost;
}

// Static list scheduling of the tasks onto `num_pairs` workers (CTA pairs): the tasks are taken head by head ((b, h) major,
// most expensive first inside a head) and each goes to the pair that is free first under the cost model above.
// All pairs therefore stream the K/V of the same head at the same time (one
// head's K, tK, V, tV stay in L2), heads overlap only at their boundaries, and because the last head ends with its
// shortest tasks the pairs finish within about one short task of each other.
//
// `head_sync`: the lists of a launch whose workers meet before every head (UmmaParams::slot_sync in per-head mode): every head
// starts from a level field (all workers free at the time the last one is), so that the wait at the rendezvous is only the
// imbalance inside one head -- about one of its shortest tasks -- instead of whatever the heads before have piled up.
void assign_workers(const std::vector<aj_task> &tasks, const Entries &ent, int32_t tile_k, int num_pairs,
                    std::vector<int32_t> &off, std::vector<int32_t> &ids, bool head_sync) {
    std::vector<int64_t> cost(tasks.size());
    for (size_t t = 0; t < tasks.size(); ++t) cost[t] = task_cost(tasks[t], ent, tile_k);
    std::vector<int32_t> order(tasks.size());
    for (size_t t = 0; t < tasks.size(); ++t) order[t] = (int32_t)t;
    std::stable_sort(order.begin(), order.end(), [&](int32_t x, int32_t y) {
        const aj_task &a = tasks[x], &c = tasks[y];
        if (a.b != c.b) return a.b < c.b;
        if (a.h != c.h) return a.h < c.h;
        return cost[x] > cost[y];
    });
    std::vector<std::vector<int32_t>> lists(num_pairs);
    std::vector<std::pair<int64_t, int>> heap;            // (-busy-until, -pair): max-heap picks the pair free first
    for (int i = 0; i < num_pairs; ++i) heap.emplace_back(0, -i);
    std::make_heap(heap.begin(), heap.end());
    int cur_b = -1, cur_h = -1;
    for (int32_t t : order) {
        if (head_sync && (tasks[t].b != cur_b || tasks[t].h != cur_h)) {
            // the workers meet before every head (the kernel's rendezvous): all of them start it at the time the last one is free
            int64_t latest = 0;
            for (auto &w : heap) latest = std::min(latest, w.first);
            for (auto &w : heap) w.first = latest;
            std::make_heap(heap.begin(), heap.end());
            cur_b = tasks[t].b; cur_h = tasks[t].h;
        }
        std::pop_heap(heap.begin(), heap.end());
        auto &top = heap.back();
        lists[-top.second].push_back(t);
        top.first -= cost[t];
        std::push_heap(heap.begin(), heap.end());
    }
    off.assign(1, 0);
    ids.clear();
    for (const auto &l : lists) { ids.insert(ids.end(), l.begin(), l.end()); off.push_back((int32_t)ids.size()); }
}

}  // namespace aj

namespace aj {

aj_status check_problem(const aj_problem *p) {
    if (!p) return aj::fail(AJ_ERR_INVALID_ARG, "problem is NULL");
    if (p->B <= 0 || p->H <= 0 || p->Nq <= 0 || p->Nk <= 0 || p->d <= 0)
        return aj::fail(AJ_ERR_INVALID_ARG, "problem: B, H, Nq, Nk, d must be > 0");
    if (p->dtype != AJ_BF16 && p->dtype != AJ_FP32) return aj::fail(AJ_ERR_INVALID_ARG, "problem: unknown dtype");
    if (!(p->scale >= 0.0f) || p->scale > 1e30f) return aj::fail(AJ_ERR_INVALID_ARG, "problem: scale must be finite and >= 0");
    return AJ_OK;
}

}  // namespace aj

extern "C" {

aj_status attn_jvp_schedule_create(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_q,
                                   int32_t tile_k, aj_schedule **out) {
    return attn_jvp_schedule_create_tiled(problem, mask, tile_q, tile_k, AJ_TILING_PER_GROUP, out);
}

aj_status attn_jvp_schedule_create_tiled(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_q,
                                         int32_t tile_k, int32_t tiling, aj_schedule **out) {
    if (!out) return aj::fail(AJ_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (aj_status st = aj::check_problem(problem)) return st;
    if (!mask) return aj::fail(AJ_ERR_INVALID_ARG, "mask is NULL");
    if (tile_q <= 0 || tile_k <= 0) return aj::fail(AJ_ERR_INVALID_ARG, "tile_q and tile_k must be > 0");
    if (tiling != AJ_TILING_PER_GROUP && tiling != AJ_TILING_PACKED) return aj::fail(AJ_ERR_INVALID_ARG, "unknown tiling");
    if (tile_q > 32767) return aj::fail(AJ_ERR_INVALID_ARG, "tile_q must be < 32768");
    aj_schedule *s = new (std::nothrow) aj_schedule();
    if (!s) return aj::fail(AJ_ERR_OOM, "out of host memory");
    try {
        s->problem = *problem; s->tile_q = tile_q; s->tile_k = tile_k; s->tiling = tiling;
        aj_status st = aj::lower_mask(*problem, *mask, s->low);
        if (st != AJ_OK) { delete s; return st; }
        if (tiling == AJ_TILING_PACKED) aj::build_tasks_packed(*problem, s->low, tile_q, tile_k, s->entries, s->tasks);
        else aj::build_tasks(*problem, s->low, tile_q, tile_k, s->entries, s->tasks);
    } catch (const std::bad_alloc &) {
        delete s;
        return aj::fail(AJ_ERR_OOM, "out of host memory");
    }
    *out = s;
    return AJ_OK;
}

aj_status attn_jvp_schedule_create_transposed(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_keys,
                                              int32_t tile_rows, aj_schedule **out) {
    return attn_jvp_schedule_create_transposed_tiled(problem, mask, tile_keys, tile_rows, AJ_TILING_PER_GROUP, out);
}

aj_status attn_jvp_schedule_create_transposed_tiled(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_keys,
                                                    int32_t tile_rows, int32_t tiling, aj_schedule **out) {
    if (!out) return aj::fail(AJ_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (aj_status st = aj::check_problem(problem)) return st;
    if (!mask) return aj::fail(AJ_ERR_INVALID_ARG, "mask is NULL");
    if (tile_keys <= 0 || tile_rows <= 0 || tile_keys > 32767) return aj::fail(AJ_ERR_INVALID_ARG, "tile sizes must be > 0 (tile_keys < 32768)");
    if (tiling != AJ_TILING_PER_GROUP && tiling != AJ_TILING_PACKED) return aj::fail(AJ_ERR_INVALID_ARG, "unknown tiling");
    aj_schedule *s = new (std::nothrow) aj_schedule();
    if (!s) return aj::fail(AJ_ERR_OOM, "out of host memory");
    try {
        aj::Lowered low;
        aj_status st = aj::lower_mask(*problem, *mask, low);
        if (st != AJ_OK) { delete s; return st; }
        s->problem = *problem;
        std::swap(s->problem.Nq, s->problem.Nk);           // the tasks' "query rows" are keys
        s->tile_q = tile_keys; s->tile_k = tile_rows; s->tiling = tiling;
        aj::transpose_lowered(*problem, low, s->low);
        if (tiling == AJ_TILING_PACKED) aj::build_tasks_packed(s->problem, s->low, tile_keys, tile_rows, s->entries, s->tasks);
        else aj::build_tasks(s->problem, s->low, tile_keys, tile_rows, s->entries, s->tasks);
    } catch (const std::bad_alloc &) {
        delete s;
        return aj::fail(AJ_ERR_OOM, "out of host memory");
    }
    *out = s;
    return AJ_OK;
}

aj_status attn_jvp_schedule_destroy(aj_schedule *sched) {
    delete sched;
    return AJ_OK;
}

aj_status attn_jvp_schedule_info(const aj_schedule *s, int32_t *num_groups, int32_t *num_ranges,
                                 int32_t *num_tasks, int64_t *pairs) {
    if (!s) return aj::fail(AJ_ERR_INVALID_ARG, "schedule is NULL");
    if (num_groups) *num_groups = (int32_t)s->low.q_begin.size();
    if (num_ranges) *num_ranges = (int32_t)s->low.ranges.size();
    if (num_tasks) *num_tasks = (int32_t)s->tasks.size();
    if (pairs) *pairs = s->low.pairs_per_head;
    return AJ_OK;
}

aj_status attn_jvp_schedule_get(const aj_schedule *s, int32_t *q_begin, int32_t *q_end, int32_t *range_offset,
                                int32_t *k_begin, int32_t *k_end, aj_task *tasks) {
    if (!s) return aj::fail(AJ_ERR_INVALID_ARG, "schedule is NULL");
    const aj::Lowered &l = s->low;
    if (q_begin) std::copy(l.q_begin.begin(), l.q_begin.end(), q_begin);
    if (q_end) std::copy(l.q_end.begin(), l.q_end.end(), q_end);
    if (range_offset) std::copy(l.range_offset.begin(), l.range_offset.end(), range_offset);
    for (size_t r = 0; r < l.ranges.size(); ++r) {
        if (k_begin) k_begin[r] = l.ranges[r].k_begin;
        if (k_end) k_end[r] = l.ranges[r].k_end;
    }
    if (tasks) std::copy(s->tasks.begin(), s->tasks.end(), tasks);
    return AJ_OK;
}

aj_status attn_jvp_schedule_entries(const aj_schedule *s, int32_t *num_entries, int32_t *k_begin, int32_t *k_end,
                                    int32_t *row_begin, int32_t *row_end) {
    if (!s) return aj::fail(AJ_ERR_INVALID_ARG, "schedule is NULL");
    const aj::Entries &e = s->entries;
    if (num_entries) *num_entries = (int32_t)e.size();
    if (k_begin) std::copy(e.k_begin.begin(), e.k_begin.end(), k_begin);
    if (k_end) std::copy(e.k_end.begin(), e.k_end.end(), k_end);
    if (row_begin) std::copy(e.row_begin.begin(), e.row_begin.end(), row_begin);
    if (row_end) std::copy(e.row_end.begin(), e.row_end.end(), row_end);
    return AJ_OK;
}

aj_status attn_jvp_schedule_entry_flags(const aj_schedule *s, int32_t *key_tangent_zero) {
    if (!s || !key_tangent_zero) return aj::fail(AJ_ERR_INVALID_ARG, "schedule or output is NULL");
    std::copy(s->entries.k_tz.begin(), s->entries.k_tz.end(), key_tangent_zero);
    return AJ_OK;
}

aj_status attn_jvp_schedule_pair_classes(const aj_schedule *s, int64_t pairs[3]) {
    if (!s || !pairs) return aj::fail(AJ_ERR_INVALID_ARG, "schedule or output is NULL");
    for (int i = 0; i < 3; ++i) pairs[i] = s->low.pair_class[i];
    return AJ_OK;
}

aj_status attn_jvp_schedule_assign(const aj_schedule *s, int32_t num_workers, int32_t *worker_offset, int32_t *task_ids) {
    if (!s) return aj::fail(AJ_ERR_INVALID_ARG, "schedule is NULL");
    if (num_workers <= 0 || !worker_offset || !task_ids) return aj::fail(AJ_ERR_INVALID_ARG, "num_workers must be > 0 and the output arrays non-NULL");
    try {
        std::vector<int32_t> off, ids;
        aj::assign_workers(s->tasks, s->entries, s->tile_k, num_workers, off, ids);
        std::copy(off.begin(), off.end(), worker_offset);
        std::copy(ids.begin(), ids.end(), task_ids);
    } catch (const std::bad_alloc &) {
        return aj::fail(AJ_ERR_OOM, "out of host memory");
    }
    return AJ_OK;
}

const char *attn_jvp_last_error(void) { return aj::last_error_cstr(); }
const char *attn_jvp_version(void) { return "attn_jvp 0.2 (sm_100a)"; }

}  // extern "C"
