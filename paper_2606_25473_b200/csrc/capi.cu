// C-ABI entry points that need CUDA: plans and the forward call (include/attn_jvp.h).
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <unordered_map>

#include "internal.hpp"
#include "kernels.hpp"

struct aj_plan {
    aj_problem problem;       // scale resolved (never 0)
    aj_mask_desc mask;        // arrays below back the pointers for AJ_MASK_RANGES
    std::vector<int32_t> m_qb, m_qe, m_off, m_kb, m_ke, m_qtz, m_ktz;
    int32_t kernel = AJ_KERNEL_SIMT;
    int32_t tiling = AJ_TILING_PER_GROUP;
    int device = 0, num_sms = 0;
    int32_t *d_counters = nullptr;
    // A schedule and its device copy.  `full` covers all B x H heads (attn_jvp_fwd); `head` is the same mask for ONE
    // (b, h) (built on first use by attn_jvp_fwd_host, which launches head by head while the copies of the
    // neighbouring heads are in flight).
    struct DevSchedule {
        aj_schedule *sched = nullptr;
        int32_t num_tasks = 0;
        aj_task *d_tasks = nullptr;
        int32_t *d_kb = nullptr, *d_ke = nullptr;
        uint32_t *d_rows = nullptr;   // per entry: row_begin | row_end << 16
        int32_t *d_pair_off = nullptr, *d_pair_ids = nullptr;   // CTA-pair kernel: host-assigned task lists
        int32_t num_pairs = 0;
        // AJ_KERNEL_UMMA_PAIR: the primal-only tasks have lists of their own (run by the forward-only kernel) and are absent
        // from the lists above
        int32_t *d_prim_off = nullptr, *d_prim_ids = nullptr;
        int32_t num_prim_pairs = 0;
        // task-slot rendezvous of the CTA-pair forward kernel (UmmaParams::slot_sync): counters and targets, one per task slot
        int32_t *d_slot_sync = nullptr, *d_slot_expect = nullptr;
        int32_t num_slots = 0, sync_per_head = 0;
    } full, head;                 // forward
    // primal backward: query tiles x key ranges (dQ) and key tiles x row ranges (dK, dV) for all B x H heads, and for ONE
    // head (attn_bwd_host)
    DevSchedule bwd_q, bwd_k, bwd_q_head, bwd_k_head;
    float *d_delta = nullptr;     // workspace of attn_bwd (bwd_alloc_bytes)
    int32_t rendezvous = AJ_RENDEZVOUS_AUTO;   // attn_jvp_plan_set_rendezvous: what the forward schedules are built for
    int32_t max_pairs = 0;                     // attn_jvp_plan_set_workers: SM pairs the CTA-pair kernels may occupy (0 = all)
    // attn_jvp_fwd_host / attn_bwd_host: device staging buffers, copy streams, one event per head and direction
    void *d_in[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // q k v tq tk tv
    void *d_out[2] = {nullptr, nullptr};                                      // o to
    void *d_bwd[4] = {nullptr, nullptr, nullptr, nullptr};                    // dout dq dk dv
    float *d_lse = nullptr;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    std::vector<cudaEvent_t> ev_in, ev_k;
    cudaEvent_t ev_begin = nullptr, ev_end = nullptr;
    // TMA descriptors the plan has encoded, one per tensor slot of a call site (the plan owns them): a slot is
    // re-encoded only when the tensor view it was encoded for changes.  `mu` guards the cache (the forward takes a const plan
    // and may be called from several host threads).
    struct MapSlot {
        const void *ptr = nullptr;
        int64_t sb = 0, sh = 0, sn = 0, rows = 0;
        int32_t box = 0, B = 0, H = 0;
        CUtensorMap map;
    };
    mutable std::mutex mu;
    mutable std::vector<MapSlot> maps;
    // 2-D maps over the backward's augmentation rows (-lse/s, -delta), one entry per call site (keyed by its first map slot:
    // attn_bwd has one, attn_bwd_host one per head, whose workspace pointers differ)
    struct AugSlot {
        const void *ptr = nullptr;
        int64_t rows = 0;
        CUtensorMap map[2];
    };
    mutable std::unordered_map<int, AugSlot> aug_maps;
    mutable int64_t map_encodes = 0, map_hits = 0;
};

namespace {

using aj::fail;

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// The driver entry point is looked up at run time so that the library links against cudart only and loads
// on machines without a driver (the CPU build box).
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

aj_status cuda_fail(cudaError_t e, const char *what) {
    return fail(AJ_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

void free_schedule(aj_plan::DevSchedule &ds) {
    cudaFree(ds.d_tasks); cudaFree(ds.d_kb); cudaFree(ds.d_ke); cudaFree(ds.d_rows);
    cudaFree(ds.d_pair_off); cudaFree(ds.d_pair_ids); cudaFree(ds.d_prim_off); cudaFree(ds.d_prim_ids);
    cudaFree(ds.d_slot_sync); cudaFree(ds.d_slot_expect);
    attn_jvp_schedule_destroy(ds.sched);
    ds = aj_plan::DevSchedule();
}

// tcgen05 kernels: the CTA-pair family (forward, forward-only, backward) for bf16 d = 128; the single-CTA forward kernel also
// for bf16 d = 64
bool pair_covers(const aj_problem &p) { return p.dtype == AJ_BF16 && p.d == 128; }
bool umma_covers(const aj_problem &p) { return p.dtype == AJ_BF16 && (p.d == 128 || p.d == 64); }

bool is_pair(int32_t kernel) { return kernel == AJ_KERNEL_UMMA_PAIR || kernel == AJ_KERNEL_UMMA_PAIR_ONE; }
bool is_umma(int32_t kernel) { return kernel == AJ_KERNEL_UMMA || is_pair(kernel); }
// bf16 d = 64: the single-CTA tcgen05 kernels
int32_t auto_kernel(const aj_problem &p) { return pair_covers(p) ? AJ_KERNEL_UMMA_PAIR : umma_covers(p) ? AJ_KERNEL_UMMA : AJ_KERNEL_SIMT; }

// The tcgen05 kernels tile queries on a global grid (no rows wasted at group ends); the SIMT kernel per group.
int32_t default_tiling(int32_t kernel) { return is_umma(kernel) ? AJ_TILING_PACKED : AJ_TILING_PER_GROUP; }


// Build the schedule of `prob` (the plan's problem, or one head of it) for `kernel` / `tiling` and upload it into `ds`
// (left unchanged on failure).
aj_status upload_schedule(aj_plan *p, aj_schedule *s, int32_t kernel, aj_plan::DevSchedule &ds, int workers = 0, bool rendezvous = false);

aj_status build_schedule(aj_plan *p, const aj_problem &prob, int32_t kernel, int32_t tiling, aj_plan::DevSchedule &ds) {
    const int tq = is_pair(kernel) ? aj::UMMA_PAIR_TILE_Q : kernel == AJ_KERNEL_UMMA ? aj::UMMA_TILE_Q : aj::SIMT_TILE_Q;
    const int tk = is_umma(kernel) ? aj::UMMA_TILE_K : aj::SIMT_TILE_K;
    if (is_pair(kernel) && tiling != AJ_TILING_PACKED)
        return fail(AJ_ERR_UNSUPPORTED, "the CTA-pair tcgen05 kernel only supports packed tiling");
    if (kernel == AJ_KERNEL_SIMT && tiling != AJ_TILING_PER_GROUP)
        return fail(AJ_ERR_UNSUPPORTED, "the SIMT kernel only supports per-group tiling");
    aj_schedule *s = nullptr;
    if (aj_status st = attn_jvp_schedule_create_tiled(&prob, &p->mask, tq, tk, tiling, &s)) return st;
    // the single-CTA tcgen05 kernel: one host-assigned, head-major task list per SM (the CTA-pair kernels get one per SM pair)
    return upload_schedule(p, s, kernel, ds, kernel == AJ_KERNEL_UMMA ? p->num_sms : 0, /*rendezvous=*/true);
}

// Uploads `s` (owned by `ds` afterwards; destroyed on failure, `ds` then unchanged).
// workers > 0: also assign the tasks to that many persistent workers (head-major lists, see assign_workers).
// rendezvous: the schedule is for the forward CTA-pair kernel, whose producers can meet per task slot / per head (long sequences).
aj_status upload_schedule(aj_plan *p, aj_schedule *s, int32_t kernel, aj_plan::DevSchedule &ds, int workers, bool rendezvous) {
    const size_t nt = s->tasks.size(), nr = s->entries.size();
    std::vector<uint32_t> rows(nr);
    for (size_t r = 0; r < nr; ++r)   // row_begin | row_end << 16 (both < 32768) | key-tangents-zero << 31
        rows[r] = (uint32_t)s->entries.row_begin[r] | ((uint32_t)s->entries.row_end[r] << 16) | (s->entries.k_tz[r] ? 0x80000000u : 0u);
    std::vector<int32_t> pair_off, pair_ids, prim_off, prim_ids;
    int num_pairs = 0, num_prim_pairs = 0;
    // tasks [ids] of the schedule onto `want` workers (fewer if there are fewer tasks); ids refer to s->tasks
    bool head_sync = false;            // the pairs meet before every head (CTA-pair forward kernel, see below)
    auto assign = [&](const std::vector<int32_t> &ids, int want, std::vector<int32_t> &off, std::vector<int32_t> &out, bool sync) {
        std::vector<aj_task> sub;
        for (int32_t t : ids) sub.push_back(s->tasks[t]);
        const int n = (int)std::min<size_t>(std::max(want, 1), std::max<size_t>(sub.size(), 1));
        aj::assign_workers(sub, s->entries, s->tile_k, n, off, out, sync);
        for (int32_t &t : out) t = ids[t];
        return n;
    };
    if (is_pair(kernel) || workers > 0) {
        const int all_pairs = std::max(p->num_sms / 2, 1);
        const int want = workers > 0 ? workers : p->max_pairs > 0 ? std::min(p->max_pairs, all_pairs) : all_pairs;
        std::vector<int32_t> general, primal;
        for (size_t t = 0; t < nt; ++t)
            ((kernel == AJ_KERNEL_UMMA_PAIR && (s->tasks[t].flags & AJ_TASK_PRIMAL_ONLY)) ? primal : general).push_back((int32_t)t);
        // Per-head rendezvous (kernel_umma_pair_sm100.cu, UmmaParams::slot_sync with sync_per_head): for the forward CTA-pair kernel when
        // the tasks of a launch differ in cost (equal ones get the task-slot rendezvous below) and the longest key stream of a task
        // is larger than what L2 keeps for all pairs (K, tK, V, tV rows of 2 d bytes each).  attn_jvp_plan_set_rendezvous forces
        // it on (PER_HEAD) or off (OFF, PER_SLOT).
        if (rendezvous && is_pair(kernel) && workers == 0 && !general.empty()) {
            int32_t tmin = INT32_MAX, tmax = 0;
            for (int32_t t : general) { tmin = std::min(tmin, s->tasks[t].num_kv_tiles); tmax = std::max(tmax, s->tasks[t].num_kv_tiles); }
            head_sync = tmin != tmax && (double)tmax * s->tile_k * 4.0 * p->problem.d * 2.0 > 48e6;
            if (p->rendezvous != AJ_RENDEZVOUS_AUTO) head_sync = p->rendezvous == AJ_RENDEZVOUS_PER_HEAD && tmax > 0;
        }
        num_pairs = assign(general, want, pair_off, pair_ids, head_sync);
        if (general.empty()) num_pairs = 0;
        if (!primal.empty()) num_prim_pairs = assign(primal, want, prim_off, prim_ids, false);
    }
    // Task-slot rendezvous (kernel_umma_pair_sm100.cu): only where it costs nothing and pays -- every task of the launch has the same
    // cost (so the pairs would start each slot together anyway), the lists are long enough for the drift to build up, and one
    // task's key stream is larger than what L2 keeps (K, tK, V, tV rows of 2 d bytes each).  AJ_RENDEZVOUS_PER_SLOT asks for it
    // on any schedule of the CTA-pair forward kernel that has no primal-only lists (the wait is bounded, so it is always safe).
    std::vector<int32_t> slot_expect;
    if (rendezvous && is_pair(kernel) && workers == 0 && num_pairs > 1 && num_prim_pairs == 0 && !pair_ids.empty() &&
        (p->rendezvous == AJ_RENDEZVOUS_AUTO || p->rendezvous == AJ_RENDEZVOUS_PER_SLOT)) {
        const aj_task &t0 = s->tasks[pair_ids[0]];
        bool uniform = t0.num_kv_tiles > 0;
        for (int32_t t : pair_ids) uniform = uniform && s->tasks[t].num_kv_tiles == t0.num_kv_tiles && s->tasks[t].flags == t0.flags;
        int max_len = 0;
        for (int w = 0; w < num_pairs; ++w) max_len = std::max(max_len, pair_off[w + 1] - pair_off[w]);
        const double stream_bytes = (double)t0.num_kv_tiles * s->tile_k * 4.0 * p->problem.d * 2.0;
        if (p->rendezvous == AJ_RENDEZVOUS_PER_SLOT || (uniform && max_len >= 16 && stream_bytes > 48e6)) {
            slot_expect.assign(max_len, 0);                    // target of slot i: the pairs whose i-th task streams any keys
            for (int w = 0; w < num_pairs; ++w)                // (the producer skips key-less tasks without arriving)
                for (int i = 0; i < pair_off[w + 1] - pair_off[w]; ++i)
                    if (s->tasks[pair_ids[pair_off[w] + i]].num_kv_tiles > 0) ++slot_expect[i];
        }
    }
    int32_t sync_per_head = 0;
    if (head_sync && num_pairs > 1) {       // tasks of different cost: the pairs meet before every head; target = the pairs that have a task in it
        slot_expect.assign((size_t)s->problem.B * s->problem.H, 0);
        for (int w = 0; w < num_pairs; ++w) {
            int prev = -1;
            for (int i = pair_off[w]; i < pair_off[w + 1]; ++i) {
                const aj_task &t = s->tasks[pair_ids[i]];
                if (t.num_kv_tiles == 0) continue;
                const int hd = t.b * s->problem.H + t.h;
                if (hd != prev) { ++slot_expect[hd]; prev = hd; }
            }
        }
        sync_per_head = 1;
    }
    aj_task *d_tasks = nullptr;
    int32_t *d_slot_sync = nullptr, *d_slot_expect = nullptr;
    int32_t *d_kb = nullptr, *d_ke = nullptr, *d_pair_off = nullptr, *d_pair_ids = nullptr, *d_prim_off = nullptr, *d_prim_ids = nullptr;
    uint32_t *d_rows = nullptr;
    cudaError_t e = cudaMalloc(&d_tasks, std::max<size_t>(nt, 1) * sizeof(aj_task));
    auto up = [&](const std::vector<int32_t> &h, int32_t **d) {
        if (e == cudaSuccess) e = cudaMalloc(d, std::max<size_t>(h.size(), 1) * sizeof(int32_t));
        if (e == cudaSuccess && !h.empty()) e = cudaMemcpy(*d, h.data(), h.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    };
    if (num_pairs) { up(pair_off, &d_pair_off); up(pair_ids, &d_pair_ids); }
    if (num_prim_pairs) { up(prim_off, &d_prim_off); up(prim_ids, &d_prim_ids); }
    if (!slot_expect.empty()) {
        up(slot_expect, &d_slot_expect);
        if (e == cudaSuccess) e = cudaMalloc(&d_slot_sync, slot_expect.size() * sizeof(int32_t));
    }
    if (e == cudaSuccess) e = cudaMalloc(&d_kb, std::max<size_t>(nr, 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&d_ke, std::max<size_t>(nr, 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&d_rows, std::max<size_t>(nr, 1) * sizeof(uint32_t));
    if (e == cudaSuccess && nt) e = cudaMemcpy(d_tasks, s->tasks.data(), nt * sizeof(aj_task), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nr) e = cudaMemcpy(d_kb, s->entries.k_begin.data(), nr * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nr) e = cudaMemcpy(d_ke, s->entries.k_end.data(), nr * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nr) e = cudaMemcpy(d_rows, rows.data(), nr * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(d_tasks); cudaFree(d_kb); cudaFree(d_ke); cudaFree(d_rows); cudaFree(d_pair_off); cudaFree(d_pair_ids);
        cudaFree(d_prim_off); cudaFree(d_prim_ids); cudaFree(d_slot_sync); cudaFree(d_slot_expect);
        attn_jvp_schedule_destroy(s);
        return e == cudaErrorMemoryAllocation ? fail(AJ_ERR_OOM, "out of device memory for the schedule") : cuda_fail(e, "schedule upload");
    }
    free_schedule(ds);
    ds.sched = s; ds.num_tasks = (int32_t)nt;
    ds.d_tasks = d_tasks; ds.d_kb = d_kb; ds.d_ke = d_ke; ds.d_rows = d_rows;
    ds.d_pair_off = d_pair_off; ds.d_pair_ids = d_pair_ids; ds.num_pairs = num_pairs;
    ds.d_prim_off = d_prim_off; ds.d_prim_ids = d_prim_ids; ds.num_prim_pairs = num_prim_pairs;
    ds.d_slot_sync = d_slot_sync; ds.d_slot_expect = d_slot_expect; ds.num_slots = (int32_t)slot_expect.size();
    ds.sync_per_head = sync_per_head;
    return AJ_OK;
}

// (Re)build the plan's schedule for `kernel` / `tiling`; the per-head schedule is rebuilt on its next use.
aj_status install_schedule(aj_plan *p, int32_t kernel, int32_t tiling) {
    if (aj_status st = build_schedule(p, p->problem, kernel, tiling, p->full)) return st;
    free_schedule(p->head);
    free_schedule(p->bwd_q);      // their tile sizes follow the kernel family
    free_schedule(p->bwd_k);
    free_schedule(p->bwd_q_head);
    free_schedule(p->bwd_k_head);
    p->kernel = kernel; p->tiling = tiling;
    return AJ_OK;
}

// `output`: the kernels write every element once, so heads / batches must not alias.  Inputs may be broadcast over heads or
// batches with a zero stride on the plain-FMA kernels; the TMA tensor maps of the tcgen05 kernels cannot express it
// (`tma` = the call will build tensor maps).
aj_status check_tensor(const aj_tensor *t, const char *name, const aj_problem &p, bool output, bool tma) {
    if (!t || !t->ptr) return fail(AJ_ERR_INVALID_ARG, std::string(name) + " is NULL");
    if ((uintptr_t)t->ptr % 16 != 0) return fail(AJ_ERR_INVALID_ARG, std::string(name) + ": pointer must be 16-byte aligned");
    if (t->stride_n < p.d || t->stride_n % 8 || t->stride_h % 8 || t->stride_b % 8 || t->stride_h < 0 || t->stride_b < 0)
        return fail(AJ_ERR_INVALID_ARG, std::string(name) + ": strides must be multiples of 8 elements with stride_n >= d");
    const bool bcast = (p.H > 1 && t->stride_h == 0) || (p.B > 1 && t->stride_b == 0);
    if (bcast && output) return fail(AJ_ERR_INVALID_ARG, std::string(name) + ": an output tensor must not alias heads or batches (zero stride)");
    if (bcast && tma) return fail(AJ_ERR_UNSUPPORTED, std::string(name) + ": zero head / batch strides (broadcast inputs) are not supported by the tcgen05 kernels");
    return AJ_OK;
}

aj_status check_device(const aj_plan *p) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev != p->device)
        return fail(AJ_ERR_INVALID_ARG, "the current CUDA device (" + std::to_string(dev) + ") is not the plan's device (" + std::to_string(p->device) + ")");
    return AJ_OK;
}

aj_status encode_map_raw(CUtensorMap *map, const aj_tensor &t, const aj_problem &p, int64_t n_rows, int box_rows) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return fail(AJ_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
    // dims innermost first: d, N, H, B.  A size-1 dimension still needs a legal (non-zero, 16-byte multiple) stride, which is
    // never used to address anything; a zero stride over a dimension > 1 was rejected by check_tensor.
    cuuint64_t dims[4] = {(cuuint64_t)p.d, (cuuint64_t)n_rows, (cuuint64_t)p.H, (cuuint64_t)p.B};
    auto bytes = [](int64_t elems, int dim) { return (cuuint64_t)(dim == 1 ? std::max<int64_t>(elems, 8) : elems) * 2; };
    cuuint64_t strides[3] = {bytes(t.stride_n, 0), bytes(t.stride_h, p.H), bytes(t.stride_b, p.B)};
    cuuint32_t box[4] = {64, (cuuint32_t)box_rows, 1, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, t.ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(AJ_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r));
    return AJ_OK;
}

// The tensor map of `t` for call-site slot `slot`: from the plan's cache if the slot was encoded for the same view.
aj_status encode_map(const aj_plan *plan, int slot, CUtensorMap *map, const aj_tensor &t, const aj_problem &p, int64_t n_rows, int box_rows) {
    std::lock_guard<std::mutex> lock(plan->mu);
    if ((size_t)slot >= plan->maps.size()) plan->maps.resize(slot + 1);
    aj_plan::MapSlot &m = plan->maps[slot];
    if (m.ptr == t.ptr && m.sb == t.stride_b && m.sh == t.stride_h && m.sn == t.stride_n && m.rows == n_rows && m.box == box_rows &&
        m.B == p.B && m.H == p.H) {
        *map = m.map;
        ++plan->map_hits;
        return AJ_OK;
    }
    if (aj_status st = encode_map_raw(&m.map, t, p, n_rows, box_rows)) { m.ptr = nullptr; return st; }
    m.ptr = t.ptr; m.sb = t.stride_b; m.sh = t.stride_h; m.sn = t.stride_n; m.rows = n_rows; m.box = box_rows; m.B = p.B; m.H = p.H;
    *map = m.map;
    ++plan->map_encodes;
    return AJ_OK;
}
// call-site slots of the cache
enum { SLOT_FWD = 0, SLOT_BWD = 8, SLOT_HEAD = 16, SLOTS_PER_HEAD = 16 };   // per head: 6 forward + 8 backward maps

}  // namespace

extern "C" {

aj_status attn_jvp_plan_create(const aj_problem *problem, const aj_mask_desc *mask, aj_plan **out) {
    if (!out) return fail(AJ_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (aj_status st = aj::check_problem(problem)) return st;
    if (!mask) return fail(AJ_ERR_INVALID_ARG, "mask is NULL");
    if (problem->d != 64 && problem->d != 128) return fail(AJ_ERR_UNSUPPORTED, "d must be 64 or 128");
    aj_plan *p = new (std::nothrow) aj_plan();
    if (!p) return fail(AJ_ERR_OOM, "out of host memory");
    aj_status st = AJ_OK;
    try {
        p->problem = *problem;
        if (p->problem.scale == 0.0f) p->problem.scale = 1.0f / std::sqrt((float)problem->d);
        p->mask = *mask;
        if (mask->kind == AJ_MASK_RANGES && mask->num_groups > 0) {
            if (!mask->q_begin || !mask->q_end || !mask->range_offset) { delete p; return fail(AJ_ERR_INVALID_ARG, "ranges mask: null group arrays"); }
            const int ng = mask->num_groups, nr = mask->range_offset[ng];
            if (nr < 0 || (nr > 0 && (!mask->k_begin || !mask->k_end))) { delete p; return fail(AJ_ERR_INVALID_ARG, "ranges mask: null range arrays"); }
            p->m_qb.assign(mask->q_begin, mask->q_begin + ng);
            p->m_qe.assign(mask->q_end, mask->q_end + ng);
            p->m_off.assign(mask->range_offset, mask->range_offset + ng + 1);
            p->m_kb.assign(mask->k_begin, mask->k_begin + nr);
            p->m_ke.assign(mask->k_end, mask->k_end + nr);
            p->mask.q_begin = p->m_qb.data(); p->mask.q_end = p->m_qe.data(); p->mask.range_offset = p->m_off.data();
            p->mask.k_begin = p->m_kb.data(); p->mask.k_end = p->m_ke.data();
            if (mask->q_tangent_zero) { p->m_qtz.assign(mask->q_tangent_zero, mask->q_tangent_zero + ng); p->mask.q_tangent_zero = p->m_qtz.data(); }
            if (mask->k_tangent_zero) { p->m_ktz.assign(mask->k_tangent_zero, mask->k_tangent_zero + nr); p->mask.k_tangent_zero = p->m_ktz.data(); }
        } else {
            p->mask.q_tangent_zero = p->mask.k_tangent_zero = nullptr;
        }
        cudaError_t e = cudaGetDevice(&p->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, p->device);
        if (e != cudaSuccess) { delete p; return cuda_fail(e, "no usable CUDA device"); }
        e = cudaMalloc(&p->d_counters, 4 * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMemset(p->d_counters, 0, 4 * sizeof(int32_t));
        if (e != cudaSuccess) { delete p; return cuda_fail(e, "counter allocation"); }
        const int32_t kernel = auto_kernel(p->problem);
        st = install_schedule(p, kernel, default_tiling(kernel));
    } catch (const std::bad_alloc &) {
        st = fail(AJ_ERR_OOM, "out of host memory");
    }
    if (st != AJ_OK) { attn_jvp_plan_destroy(p); return st; }
    *out = p;
    return AJ_OK;
}

aj_status attn_jvp_plan_destroy(aj_plan *p) {
    if (!p) return AJ_OK;
    free_schedule(p->full);
    free_schedule(p->head);
    free_schedule(p->bwd_q);
    free_schedule(p->bwd_k);
    free_schedule(p->bwd_q_head);
    free_schedule(p->bwd_k_head);
    cudaFree(p->d_delta);
    cudaFree(p->d_counters);
    for (void *x : p->d_in) cudaFree(x);
    for (void *x : p->d_out) cudaFree(x);
    for (void *x : p->d_bwd) cudaFree(x);
    cudaFree(p->d_lse);
    for (cudaEvent_t e : p->ev_in) cudaEventDestroy(e);
    for (cudaEvent_t e : p->ev_k) cudaEventDestroy(e);
    if (p->ev_begin) cudaEventDestroy(p->ev_begin);
    if (p->ev_end) cudaEventDestroy(p->ev_end);
    if (p->s_in) cudaStreamDestroy(p->s_in);
    if (p->s_out) cudaStreamDestroy(p->s_out);
    delete p;
    return AJ_OK;
}

aj_status attn_jvp_plan_info(const aj_plan *p, int64_t *pairs, int32_t *num_tasks) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (pairs) *pairs = p->full.sched->low.pairs_per_head;
    if (num_tasks) *num_tasks = p->full.num_tasks;
    return AJ_OK;
}

aj_status attn_jvp_plan_pair_classes(const aj_plan *p, int64_t pairs[3]) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    return attn_jvp_schedule_pair_classes(p->full.sched, pairs);
}

aj_status attn_jvp_plan_set_kernel(aj_plan *p, int32_t kernel) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (kernel == AJ_KERNEL_AUTO) kernel = auto_kernel(p->problem);
    if (kernel != AJ_KERNEL_SIMT && !is_umma(kernel)) return fail(AJ_ERR_INVALID_ARG, "unknown kernel");
    if (is_umma(kernel) && !umma_covers(p->problem)) return fail(AJ_ERR_UNSUPPORTED, "the tcgen05 kernels need bf16 inputs");
    if (is_pair(kernel) && !pair_covers(p->problem)) return fail(AJ_ERR_UNSUPPORTED, "the CTA-pair tcgen05 kernels need d = 128 (bf16 d = 64 runs AJ_KERNEL_UMMA)");
    if (kernel == p->kernel) return AJ_OK;
    return install_schedule(p, kernel, default_tiling(kernel));
}

aj_status attn_jvp_plan_set_tiling(aj_plan *p, int32_t tiling) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (tiling != AJ_TILING_PER_GROUP && tiling != AJ_TILING_PACKED) return fail(AJ_ERR_INVALID_ARG, "unknown tiling");
    if (tiling == p->tiling) return AJ_OK;
    return install_schedule(p, p->kernel, tiling);
}

aj_status attn_jvp_plan_set_rendezvous(aj_plan *p, int32_t mode) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (mode != AJ_RENDEZVOUS_AUTO && mode != AJ_RENDEZVOUS_OFF && mode != AJ_RENDEZVOUS_PER_SLOT && mode != AJ_RENDEZVOUS_PER_HEAD)
        return fail(AJ_ERR_INVALID_ARG, "unknown rendezvous mode");
    if (mode == p->rendezvous) return AJ_OK;
    const int32_t old = p->rendezvous;
    p->rendezvous = mode;
    if (aj_status st = install_schedule(p, p->kernel, p->tiling)) { p->rendezvous = old; return st; }
    return AJ_OK;
}

aj_status attn_jvp_plan_set_workers(aj_plan *p, int32_t num_pairs) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (num_pairs < 0) return fail(AJ_ERR_INVALID_ARG, "num_pairs must be >= 0 (0 = every SM pair of the device)");
    if (num_pairs == p->max_pairs) return AJ_OK;
    const int32_t old = p->max_pairs;
    p->max_pairs = num_pairs;
    // forward lists now; the backward lists are rebuilt on the next attn_bwd (install_schedule drops them)
    if (aj_status st = install_schedule(p, p->kernel, p->tiling)) { p->max_pairs = old; return st; }
    return AJ_OK;
}

aj_status attn_jvp_plan_workers(const aj_plan *p, int32_t *num_pairs, int32_t *num_primal_pairs) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (num_pairs) *num_pairs = p->full.num_pairs;
    if (num_primal_pairs) *num_primal_pairs = p->full.num_prim_pairs;
    return AJ_OK;
}

aj_status attn_jvp_plan_rendezvous(const aj_plan *p, int32_t *in_effect) {
    if (!p || !in_effect) return fail(AJ_ERR_INVALID_ARG, "plan or in_effect is NULL");
    *in_effect = p->full.num_slots == 0 ? AJ_RENDEZVOUS_OFF : p->full.sync_per_head ? AJ_RENDEZVOUS_PER_HEAD : AJ_RENDEZVOUS_PER_SLOT;
    return AJ_OK;
}

aj_status attn_jvp_plan_kernel(const aj_plan *p, int32_t *kernel, int32_t *launches) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (kernel) *kernel = p->kernel;
    if (launches) *launches = p->full.num_tasks == 0 ? 0 : is_pair(p->kernel) ? (p->full.num_pairs > 0) + (p->full.num_prim_pairs > 0) : 1;
    return AJ_OK;
}

aj_status attn_jvp_plan_device_status(aj_plan *p, int32_t *code) {
    if (!p || !code) return fail(AJ_ERR_INVALID_ARG, "plan or code is NULL");
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(code, p->d_counters + 2, sizeof(int32_t), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && *code != 0) e = cudaMemset(p->d_counters, 0, 4 * sizeof(int32_t));
    if (e != cudaSuccess) return cuda_fail(e, "device status");
    return AJ_OK;
}

}  // extern "C"

namespace {

// One kernel launch over the tasks of `ds`, which were built for a [B, H] problem (the plan's, or B = H = 1 with the
// tensor views already moved to the head they address).  `slot`: first of the six tensor-map cache slots of the call site.
aj_status launch_schedule(const aj_plan *p, const aj_plan::DevSchedule &ds, int32_t B, int32_t H, const aj_tensor *const ts[8],
                          float *lse, float *tlse, cudaStream_t stream, int slot) {
    aj_problem pr = p->problem;
    pr.B = B; pr.H = H;
    if (ds.num_tasks == 0) return AJ_OK;
    cudaError_t e;
    // AJ_TANGENT_NONE plans: every kernel ignores tq, tk, tv (they may be NULL), writes tO = 0 where `to` is given and
    // tlse = 0 (the tensor maps of the absent tangents alias the primals so that they stay valid)
    const bool none = p->mask.tangent_zero == AJ_TANGENT_NONE;
    if (is_umma(p->kernel)) {
        aj::UmmaParams prm;
        std::memset(&prm, 0, sizeof(prm));
        aj_status st;
        const aj_tensor *tq = (none || !ts[3]) ? ts[0] : ts[3], *tk = (none || !ts[4]) ? ts[1] : ts[4], *tv = (none || !ts[5]) ? ts[2] : ts[5];
        if ((st = encode_map(p, slot + 0, &prm.tm_q, *ts[0], pr, pr.Nq, aj::UMMA_TILE_Q))) return st;
        if ((st = encode_map(p, slot + 1, &prm.tm_tq, *tq, pr, pr.Nq, aj::UMMA_TILE_Q))) return st;
        if ((st = encode_map(p, slot + 2, &prm.tm_k, *ts[1], pr, pr.Nk, aj::UMMA_TILE_K))) return st;
        if ((st = encode_map(p, slot + 3, &prm.tm_tk, *tk, pr, pr.Nk, aj::UMMA_TILE_K))) return st;
        if ((st = encode_map(p, slot + 4, &prm.tm_v, *ts[2], pr, pr.Nk, aj::UMMA_TILE_K))) return st;
        if ((st = encode_map(p, slot + 5, &prm.tm_tv, *tv, pr, pr.Nk, aj::UMMA_TILE_K))) return st;
        prm.o = *ts[6]; prm.lse = lse; prm.tlse = tlse;
        if (ts[7]) prm.to = *ts[7];
        prm.tasks = ds.d_tasks; prm.k_begin = ds.d_kb; prm.k_end = ds.d_ke; prm.rows = ds.d_rows; prm.counters = p->d_counters;
        prm.num_tasks = ds.num_tasks; prm.H = pr.H; prm.Nq = pr.Nq;
        prm.scale = pr.scale; prm.scale_log2 = pr.scale * 1.4426950408889634f;
        prm.pair_off = ds.d_pair_off; prm.pair_ids = ds.d_pair_ids;
        if (is_pair(p->kernel)) {
            e = cudaSuccess;
            if (ds.num_prim_pairs > 0) {                 // the tasks without tangents: the forward-only kernel, lists of their own
                aj::UmmaParams pp = prm;
                pp.pair_off = ds.d_prim_off; pp.pair_ids = ds.d_prim_ids;
                e = aj::launch_umma_pair_fwd(pp, ds.num_prim_pairs, stream);
            }
            if (e == cudaSuccess && ds.num_pairs > 0) {
                if (ds.num_slots > 0) {
                    prm.slot_sync = ds.d_slot_sync; prm.slot_expect = ds.d_slot_expect; prm.sync_per_head = ds.sync_per_head;
                    e = cudaMemsetAsync(ds.d_slot_sync, 0, ds.num_slots * sizeof(int32_t), stream);
                }
                if (e == cudaSuccess) e = aj::launch_umma_pair(prm, ds.num_pairs, stream);
            }
        } else {
            e = aj::launch_umma(prm, pr.d, none, ds.num_pairs, stream);
        }
    } else {
        aj::SimtParams prm;
        std::memset(&prm, 0, sizeof(prm));
        prm.q = *ts[0]; prm.k = *ts[1]; prm.v = *ts[2]; prm.o = *ts[6];
        if (!none) { prm.tq = *ts[3]; prm.tk = *ts[4]; prm.tv = *ts[5]; }
        if (ts[7]) prm.to = *ts[7];
        prm.no_tangents = none ? 1 : 0;
        prm.lse = lse; prm.tlse = tlse; prm.tasks = ds.d_tasks; prm.k_begin = ds.d_kb; prm.k_end = ds.d_ke;
        prm.H = pr.H; prm.Nq = pr.Nq; prm.scale = pr.scale;
        e = aj::launch_simt(prm, pr.dtype, pr.d, ds.num_tasks, stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
    return AJ_OK;
}

}  // namespace

extern "C" {

aj_status attn_jvp_fwd_tl(const aj_plan *p, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v, const aj_tensor *tq,
                          const aj_tensor *tk, const aj_tensor *tv, const aj_tensor *o, const aj_tensor *to, float *lse,
                          float *tlse, void *cuda_stream) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (aj_status st = check_device(p)) return st;
    const aj_problem &pr = p->problem;
    const aj_tensor *ts[8] = {q, k, v, tq, tk, tv, o, to};
    const char *names[8] = {"q", "k", "v", "tq", "tk", "tv", "o", "to"};
    const bool may_omit = p->mask.tangent_zero == AJ_TANGENT_NONE;
    for (int i = 0; i < 8; ++i) {
        const bool tangent = (i >= 3 && i <= 5) || i == 7;
        if (tangent && may_omit && !ts[i]) continue;
        if (aj_status st = check_tensor(ts[i], names[i], pr, i >= 6, is_umma(p->kernel))) return st;
    }
    if (lse && (uintptr_t)lse % 4 != 0) return fail(AJ_ERR_INVALID_ARG, "lse: pointer must be 4-byte aligned");
    if (tlse && (uintptr_t)tlse % 4 != 0) return fail(AJ_ERR_INVALID_ARG, "tlse: pointer must be 4-byte aligned");
    return launch_schedule(p, p->full, pr.B, pr.H, ts, lse, tlse, (cudaStream_t)cuda_stream, SLOT_FWD);
}

aj_status attn_jvp_fwd(const aj_plan *p, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v, const aj_tensor *tq,
                       const aj_tensor *tk, const aj_tensor *tv, const aj_tensor *o, const aj_tensor *to, float *lse,
                       void *cuda_stream) {
    return attn_jvp_fwd_tl(p, q, k, v, tq, tk, tv, o, to, lse, nullptr, cuda_stream);
}

aj_status attn_fwd(const aj_plan *p, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v, const aj_tensor *o, float *lse,
                   void *cuda_stream) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (p->mask.tangent_zero != AJ_TANGENT_NONE) return fail(AJ_ERR_INVALID_ARG, "attn_fwd needs a plan whose mask says AJ_TANGENT_NONE");
    return attn_jvp_fwd(p, q, k, v, nullptr, nullptr, nullptr, o, nullptr, lse, cuda_stream);
}

}  // extern "C"

namespace {

// Which kernels the backward runs: plain FMA (fp32, d = 64, or a plan forced to SIMT), the single-CTA tcgen05 kernel (a plan
// forced to AJ_KERNEL_UMMA), or CTA pairs (default).
enum BwdFamily { BWD_SIMT = 0, BWD_UMMA = 1, BWD_PAIR = 2 };
BwdFamily bwd_family(const aj_plan *p) {
    if (!umma_covers(p->problem) || p->kernel == AJ_KERNEL_SIMT) return BWD_SIMT;
    if (p->kernel == AJ_KERNEL_UMMA || !pair_covers(p->problem)) return BWD_UMMA;    // bf16 d = 64: the single-CTA kernels
    return BWD_PAIR;
}

// The backward schedules of `prob` (the plan's problem, or one head of it): query tiles x key ranges (dQ) and key tiles x
// row ranges (dK, dV; the transposed mask), tiled for the kernel family that will run; built and uploaded on first use.
// The tangent promises of the mask do not concern the backward: its schedules are built from the DENSE descriptor.
aj_status ensure_bwd_schedules(aj_plan *p, const aj_problem &prob, BwdFamily fam, aj_plan::DevSchedule &bq, aj_plan::DevSchedule &bk) {
    const int tile_s = fam == BWD_PAIR ? aj::UMMA_PAIR_TILE_Q : fam == BWD_UMMA ? aj::UMMA_TILE_Q : aj::SIMT_TILE_Q;
    const int tile_m = fam == BWD_SIMT ? aj::SIMT_TILE_K : aj::UMMA_TILE_K;
    const int32_t tiling = fam == BWD_PAIR ? AJ_TILING_PACKED : AJ_TILING_PER_GROUP;
    const int32_t kernel = fam == BWD_PAIR ? AJ_KERNEL_UMMA_PAIR : AJ_KERNEL_SIMT;     // what upload_schedule lays the lists out for
    const int workers = fam == BWD_UMMA ? p->num_sms : 0;                               // single-CTA kernel: one list per SM
    aj_mask_desc dense = p->mask;
    dense.tangent_zero = AJ_TANGENT_DENSE;
    dense.q_tangent_zero = dense.k_tangent_zero = nullptr;
    if (!bq.sched) {
        aj_schedule *s = nullptr;
        if (aj_status st = attn_jvp_schedule_create_tiled(&prob, &dense, tile_s, tile_m, tiling, &s)) return st;
        if (aj_status st = upload_schedule(p, s, kernel, bq, workers)) return st;
    }
    if (!bk.sched) {
        aj_schedule *s = nullptr;
        if (aj_status st = attn_jvp_schedule_create_transposed_tiled(&prob, &dense, tile_s, tile_m, tiling, &s)) return st;
        if (aj_status st = upload_schedule(p, s, kernel, bk, workers)) return st;
    }
    return AJ_OK;
}

// Backward workspace of `rows` = B * H * Nq query rows: [delta: rows floats] for the SIMT and single-CTA kernels; for the CTA
// pairs [{lse log2e, delta}: rows float2, padded to 16 B][aug rows of -lse/s: rows x 32 B][aug rows of -delta: rows x 32 B].
size_t bwd_ld_bytes(int64_t rows) { return ((size_t)rows * 8 + 15) & ~(size_t)15; }
size_t bwd_work_bytes(int64_t rows) { return bwd_ld_bytes(rows) + (size_t)rows * 64; }
// what a plan allocates: enough for one call over all heads and for B * H per-head calls (attn_bwd_host)
size_t bwd_alloc_bytes(const aj_problem &pr) {
    return std::max(bwd_work_bytes((int64_t)pr.B * pr.H * pr.Nq), bwd_work_bytes(pr.Nq) * (size_t)pr.B * pr.H);
}

// 2-D maps over the two aug arrays ([rows][16] bf16 each, box {16, 64}); cached in the plan per call site `slot`
aj_status encode_aug_maps(const aj_plan *plan, int slot, CUtensorMap *m1, CUtensorMap *m2, const void *aug, int64_t rows) {
    std::lock_guard<std::mutex> lock(plan->mu);
    aj_plan::AugSlot &a = plan->aug_maps[slot];
    if (a.ptr != aug || a.rows != rows) {
        EncodeTiledFn fn = encode_tiled_fn();
        if (!fn) return fail(AJ_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
        for (int i = 0; i < 2; ++i) {
            cuuint64_t dims[2] = {16, (cuuint64_t)rows};
            cuuint64_t strides[1] = {32};
            cuuint32_t box[2] = {16, 64}, estr[2] = {1, 1};
            CUresult r = fn(&a.map[i], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, (char *)aug + (size_t)i * rows * 32, dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) { a.ptr = nullptr; return fail(AJ_ERR_CUDA, "cuTensorMapEncodeTiled (augmentation rows) failed with CUresult " + std::to_string((int)r)); }
        }
        a.ptr = aug; a.rows = rows;
        plan->map_encodes += 2;
    } else {
        plan->map_hits += 2;
    }
    *m1 = a.map[0]; *m2 = a.map[1];
    return AJ_OK;
}

// The kernels of one backward call over the tasks of (bq, bk), which were built for a [B, H] problem.
// ts = {q, k, v, o, dout, dq, dk, dv}; lse: [B, H, Nq] of that problem; work: bwd_work_bytes(B * H * Nq) bytes;
// `slot`: first of eight tensor-map slots.
aj_status launch_bwd(const aj_plan *p, const aj_plan::DevSchedule &bq, const aj_plan::DevSchedule &bk, int32_t B, int32_t H,
                     const aj_tensor *const ts[8], const float *lse, float *work, cudaStream_t stream, int slot) {
    aj_problem pr = p->problem;
    pr.B = B; pr.H = H;
    const BwdFamily fam = bwd_family(p);
    const aj_tensor *q = ts[0], *k = ts[1], *v = ts[2], *o = ts[3], *dout = ts[4], *dq = ts[5], *dk = ts[6], *dv = ts[7];
    aj::BwdParams prm;
    prm.q = *q; prm.k = *k; prm.v = *v; prm.o = *o; prm.dout = *dout; prm.dq = *dq; prm.dk = *dk; prm.dv = *dv;
    prm.lse = lse;
    prm.delta = fam == BWD_PAIR ? nullptr : work;
    const int64_t rows = (int64_t)pr.B * pr.H * pr.Nq;
    void *aug = (char *)work + bwd_ld_bytes(rows);
    prm.ld = fam == BWD_PAIR ? (float2 *)work : nullptr;
    prm.aug = fam == BWD_PAIR ? (uint4 *)aug : nullptr;
    prm.q_tasks = bq.d_tasks; prm.q_kb = bq.d_kb; prm.q_ke = bq.d_ke;
    prm.k_tasks = bk.d_tasks; prm.k_rb = bk.d_kb; prm.k_re = bk.d_ke;
    prm.B = pr.B; prm.H = pr.H; prm.Nq = pr.Nq; prm.scale = pr.scale;
    cudaError_t e;
    if (fam == BWD_SIMT) {
        e = aj::launch_bwd_simt(prm, pr.dtype, pr.d, bq.num_tasks, bk.num_tasks, stream);
        if (e != cudaSuccess) return cuda_fail(e, "backward kernel launch");
        return AJ_OK;
    }
    e = aj::launch_bwd_delta(prm, pr.dtype, pr.d, stream);
    if (e != cudaSuccess) return cuda_fail(e, "backward delta kernel launch");
    for (int pass = 0; pass < 2; ++pass) {
        const bool keys = pass == 1;
        const aj_plan::DevSchedule &ds = keys ? bk : bq;
        // stationary operands (128-row boxes) and streamed operands (64-row boxes) of the pass
        const aj_tensor *a1 = keys ? k : q, *a2 = keys ? v : dout, *b1 = keys ? q : k, *b2 = keys ? dout : v;
        const int64_t na = keys ? pr.Nk : pr.Nq, nb = keys ? pr.Nq : pr.Nk;
        aj_status st;
        if (fam == BWD_PAIR) {
            aj::BwdPairParams up;
            std::memset(&up, 0, sizeof(up));
            if (keys) {
                if ((st = encode_map(p, slot + 4 * pass + 0, &up.tm_a1, *a1, pr, na, aj::UMMA_TILE_Q))) return st;
                if ((st = encode_map(p, slot + 4 * pass + 1, &up.tm_a2, *a2, pr, na, aj::UMMA_TILE_Q))) return st;
                if ((st = encode_aug_maps(p, slot, &up.tm_aug1, &up.tm_aug2, aug, rows))) return st;
            }
            if ((st = encode_map(p, slot + 4 * pass + 2, &up.tm_b1, *b1, pr, nb, aj::UMMA_TILE_K))) return st;
            if ((st = encode_map(p, slot + 4 * pass + 3, &up.tm_b2, *b2, pr, nb, aj::UMMA_TILE_K))) return st;
            if (!keys) {   // the dQ pass stages half a streamed tile (32 rows) per CTA for X and Y: cache slots of the unused a1, a2
                if ((st = encode_map(p, slot + 0, &up.tm_b1h, *b1, pr, nb, aj::UMMA_TILE_K / 2))) return st;
                if ((st = encode_map(p, slot + 1, &up.tm_b2h, *b2, pr, nb, aj::UMMA_TILE_K / 2))) return st;
            }
            up.a1 = *a1; up.a2 = *a2;
            up.out1 = keys ? *dk : *dq;
            up.out2 = *dv;
            up.ld = (const float2 *)work;
            up.tasks = ds.d_tasks; up.r_begin = ds.d_kb; up.r_end = ds.d_ke; up.rows = ds.d_rows; up.err = p->d_counters + 2;
            up.pair_off = ds.d_pair_off; up.pair_ids = ds.d_pair_ids;
            up.num_tasks = ds.num_tasks; up.H = pr.H; up.Nq = pr.Nq;
            up.scale = pr.scale; up.scale_log2 = pr.scale * 1.4426950408889634f;
            e = aj::launch_bwd_umma_pair(up, keys, ds.num_pairs, stream);
        } else {
            aj::BwdUmmaParams up;
            std::memset(&up, 0, sizeof(up));
            if ((st = encode_map(p, slot + 4 * pass + 0, &up.tm_a1, *a1, pr, na, aj::UMMA_TILE_Q))) return st;
            if ((st = encode_map(p, slot + 4 * pass + 1, &up.tm_a2, *a2, pr, na, aj::UMMA_TILE_Q))) return st;
            if ((st = encode_map(p, slot + 4 * pass + 2, &up.tm_b1, *b1, pr, nb, aj::UMMA_TILE_K))) return st;
            if ((st = encode_map(p, slot + 4 * pass + 3, &up.tm_b2, *b2, pr, nb, aj::UMMA_TILE_K))) return st;
            up.a1 = *a1; up.a2 = *a2; up.Na = (int32_t)na;
            up.out1 = keys ? *dk : *dq;
            up.out2 = *dv;
            up.lse = lse; up.delta = work;
            up.tasks = ds.d_tasks; up.r_begin = ds.d_kb; up.r_end = ds.d_ke; up.err = p->d_counters + 2;
            up.cta_off = ds.d_pair_off; up.cta_ids = ds.d_pair_ids;
            up.num_tasks = ds.num_tasks; up.H = pr.H; up.Nq = pr.Nq;
            up.scale = pr.scale; up.scale_log2 = pr.scale * 1.4426950408889634f;
            e = aj::launch_bwd_umma(up, pr.d, keys, ds.num_pairs, stream);
        }
        if (e != cudaSuccess) return cuda_fail(e, "backward kernel launch");
    }
    return AJ_OK;
}

// device staging of the host-buffer calls: `n` buffers of `bytes` each, allocated on first use
aj_status ensure_staging(void **bufs, int n, const size_t *bytes) {
    for (int i = 0; i < n; ++i)
        if (!bufs[i]) {
            cudaError_t e = cudaMalloc(&bufs[i], bytes[i]);
            if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? fail(AJ_ERR_OOM, "out of device memory for staging") : cuda_fail(e, "staging allocation");
        }
    return AJ_OK;
}

aj_status ensure_copy_streams(aj_plan *p) {
    if (p->s_in) return AJ_OK;
    const int nheads = p->problem.B * p->problem.H;
    cudaError_t e = cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_begin, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_end, cudaEventDisableTiming);
    p->ev_in.assign(nheads, nullptr); p->ev_k.assign(nheads, nullptr);
    for (int i = 0; i < nheads && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_k[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) return cuda_fail(e, "copy streams / events");
    return AJ_OK;
}

}  // namespace

extern "C" {

aj_status attn_bwd(aj_plan *p, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v, const aj_tensor *o, const float *lse,
                   const aj_tensor *dout, const aj_tensor *dq, const aj_tensor *dk, const aj_tensor *dv, void *cuda_stream) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (aj_status st = check_device(p)) return st;
    const aj_problem &pr = p->problem;
    const aj_tensor *ts[8] = {q, k, v, o, dout, dq, dk, dv};
    const char *names[8] = {"q", "k", "v", "o", "dout", "dq", "dk", "dv"};
    const BwdFamily fam = bwd_family(p);
    for (int i = 0; i < 8; ++i)
        if (aj_status st = check_tensor(ts[i], names[i], pr, i >= 5, fam != BWD_SIMT)) return st;
    if (!lse || (uintptr_t)lse % 4 != 0) return fail(AJ_ERR_INVALID_ARG, "lse: NULL or misaligned");
    // first use: the two schedules and the delta workspace (synchronous host work and allocations)
    if (aj_status st = ensure_bwd_schedules(p, p->problem, fam, p->bwd_q, p->bwd_k)) return st;
    if (!p->d_delta) {
        cudaError_t e = cudaMalloc(&p->d_delta, bwd_alloc_bytes(pr));
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? fail(AJ_ERR_OOM, "out of device memory for the backward workspace") : cuda_fail(e, "workspace allocation");
    }
    return launch_bwd(p, p->bwd_q, p->bwd_k, pr.B, pr.H, ts, lse, p->d_delta, (cudaStream_t)cuda_stream, SLOT_BWD);
}

aj_status attn_bwd_host(aj_plan *p, const void *q, const void *k, const void *v, const void *o, const float *lse,
                        const void *dout, void *dq, void *dk, void *dv, void *cuda_stream) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (aj_status st = check_device(p)) return st;
    if (!q || !k || !v || !o || !lse || !dout || !dq || !dk || !dv) return fail(AJ_ERR_INVALID_ARG, "a host pointer is NULL");
    const aj_problem &pr = p->problem;
    const size_t eb = pr.dtype == AJ_BF16 ? 2 : 4;
    const int nheads = pr.B * pr.H;
    const size_t hq = (size_t)pr.Nq * pr.d * eb, hk = (size_t)pr.Nk * pr.d * eb;     // one head of a tensor
    const size_t nq_bytes = hq * nheads, nk_bytes = hk * nheads, lse_bytes = (size_t)nheads * pr.Nq * sizeof(float);
    const size_t head_work = bwd_work_bytes(pr.Nq), work_bytes = bwd_alloc_bytes(pr);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    {   // staging: q k v (shared with the forward) | o | dout dq dk dv | lse | delta / {lse log2e, delta}
        const size_t in_bytes[3] = {nq_bytes, nk_bytes, nk_bytes}, bwd_bytes[4] = {nq_bytes, nq_bytes, nk_bytes, nk_bytes};
        if (aj_status st = ensure_staging(p->d_in, 3, in_bytes)) return st;
        if (aj_status st = ensure_staging(p->d_out, 1, &nq_bytes)) return st;
        if (aj_status st = ensure_staging(p->d_bwd, 4, bwd_bytes)) return st;
        if (aj_status st = ensure_staging((void **)&p->d_lse, 1, &lse_bytes)) return st;
        if (aj_status st = ensure_staging((void **)&p->d_delta, 1, &work_bytes)) return st;
    }
    if (aj_status st = ensure_copy_streams(p)) return st;
    aj_problem one = p->problem;
    one.B = 1; one.H = 1;
    if (aj_status st = ensure_bwd_schedules(p, one, bwd_family(p), p->bwd_q_head, p->bwd_k_head)) return st;
    // Same pipeline as attn_jvp_fwd_host: head i's q, k, v, o, dout, lse go up on the copy-in stream, its three kernels run on
    // the caller's stream as soon as they have landed, its dq, dk, dv come back on the copy-out stream.
    cudaError_t e = cudaEventRecord(p->ev_begin, stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_in, p->ev_begin, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_out, p->ev_begin, 0);
    if (e != cudaSuccess) return cuda_fail(e, "stream ordering");
    const void *src[5] = {q, k, v, o, dout};
    void *dst[5] = {p->d_in[0], p->d_in[1], p->d_in[2], p->d_out[0], p->d_bwd[0]};
    void *res_d[3] = {p->d_bwd[1], p->d_bwd[2], p->d_bwd[3]};
    void *res_h[3] = {dq, dk, dv};
    for (int hd = 0; hd < nheads; ++hd) {
        for (int i = 0; i < 5 && e == cudaSuccess; ++i) {
            const size_t hb = (i == 1 || i == 2) ? hk : hq;
            e = cudaMemcpyAsync((char *)dst[i] + hd * hb, (const char *)src[i] + hd * hb, hb, cudaMemcpyHostToDevice, p->s_in);
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(p->d_lse + (size_t)hd * pr.Nq, lse + (size_t)hd * pr.Nq, pr.Nq * sizeof(float), cudaMemcpyHostToDevice, p->s_in);
        if (e == cudaSuccess) e = cudaEventRecord(p->ev_in[hd], p->s_in);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, p->ev_in[hd], 0);
        if (e != cudaSuccess) return cuda_fail(e, "host-to-device copy");
        aj_tensor t[8];
        const aj_tensor *ts[8];
        void *base[8] = {p->d_in[0], p->d_in[1], p->d_in[2], p->d_out[0], p->d_bwd[0], p->d_bwd[1], p->d_bwd[2], p->d_bwd[3]};
        for (int i = 0; i < 8; ++i) {
            const bool is_k = i == 1 || i == 2 || i >= 6;
            const int64_t n = is_k ? pr.Nk : pr.Nq;
            t[i].ptr = (char *)base[i] + hd * (is_k ? hk : hq);
            t[i].stride_n = pr.d; t[i].stride_h = n * pr.d; t[i].stride_b = n * pr.d;
            ts[i] = &t[i];
        }
        if (aj_status st = launch_bwd(p, p->bwd_q_head, p->bwd_k_head, 1, 1, ts, p->d_lse + (size_t)hd * pr.Nq,
                                      (float *)((char *)p->d_delta + hd * head_work), stream, SLOT_HEAD + hd * SLOTS_PER_HEAD + 8)) return st;
        e = cudaEventRecord(p->ev_k[hd], stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_out, p->ev_k[hd], 0);
        for (int i = 0; i < 3 && e == cudaSuccess; ++i) {
            const size_t hb = i == 0 ? hq : hk;
            e = cudaMemcpyAsync((char *)res_h[i] + hd * hb, (char *)res_d[i] + hd * hb, hb, cudaMemcpyDeviceToHost, p->s_out);
        }
        if (e != cudaSuccess) return cuda_fail(e, "device-to-host copy");
    }
    e = cudaEventRecord(p->ev_end, p->s_out);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, p->ev_end, 0);
    if (e != cudaSuccess) return cuda_fail(e, "stream ordering");
    return AJ_OK;
}

aj_status attn_jvp_fwd_host(aj_plan *p, const void *q, const void *k, const void *v, const void *tq, const void *tk,
                            const void *tv, void *o, void *to, float *lse, void *cuda_stream) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    if (aj_status st = check_device(p)) return st;
    const void *in[6] = {q, k, v, tq, tk, tv};
    const bool no_tangents = p->mask.tangent_zero == AJ_TANGENT_NONE && !tq && !tk && !tv && !to;   // forward only
    for (int i = 0; i < (no_tangents ? 3 : 6); ++i) if (!in[i]) return fail(AJ_ERR_INVALID_ARG, "a host input pointer is NULL");
    if (!o || (!to && !no_tangents)) return fail(AJ_ERR_INVALID_ARG, "a host output pointer is NULL");
    const aj_problem &pr = p->problem;
    const size_t eb = pr.dtype == AJ_BF16 ? 2 : 4;
    const int nheads = pr.B * pr.H;
    const size_t hq_bytes = (size_t)pr.Nq * pr.d * eb, hk_bytes = (size_t)pr.Nk * pr.d * eb;   // one head of a tensor
    const size_t nq_bytes = hq_bytes * nheads, nk_bytes = hk_bytes * nheads;
    const size_t lse_bytes = (size_t)nheads * pr.Nq * sizeof(float);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    {
        const size_t in_bytes[6] = {nq_bytes, nk_bytes, nk_bytes, nq_bytes, nk_bytes, nk_bytes}, out_bytes[2] = {nq_bytes, nq_bytes};
        if (aj_status st = ensure_staging(p->d_in, no_tangents ? 3 : 6, in_bytes)) return st;
        if (aj_status st = ensure_staging(p->d_out, no_tangents ? 1 : 2, out_bytes)) return st;
        if (aj_status st = ensure_staging((void **)&p->d_lse, 1, &lse_bytes)) return st;
    }
    if (aj_status st = ensure_copy_streams(p)) return st;
    cudaError_t e = cudaSuccess;
    if (!p->head.sched) {
        aj_problem one = p->problem;
        one.B = 1; one.H = 1;
        if (aj_status st = build_schedule(p, one, p->kernel, p->tiling, p->head)) return st;
    }
    // Heads are independent: head i's six slices go up on the copy-in stream, its kernel runs on the
    // caller's stream as soon as they have landed, and its O, tO, lse come back on the copy-out stream, so the copies
    // of heads i+1 and i-1 overlap the kernel of head i.  The caller's stream finally waits for the last D2H copy.
    e = cudaEventRecord(p->ev_begin, stream);                       // earlier work on `stream` may still use the staging buffers
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_in, p->ev_begin, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_out, p->ev_begin, 0);
    if (e != cudaSuccess) return cuda_fail(e, "stream ordering");
    for (int hd = 0; hd < nheads; ++hd) {
        for (int i = 0; i < (no_tangents ? 3 : 6) && e == cudaSuccess; ++i) {
            const size_t hb = (i == 0 || i == 3) ? hq_bytes : hk_bytes;
            e = cudaMemcpyAsync((char *)p->d_in[i] + hd * hb, (const char *)in[i] + hd * hb, hb, cudaMemcpyHostToDevice, p->s_in);
        }
        if (e == cudaSuccess) e = cudaEventRecord(p->ev_in[hd], p->s_in);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, p->ev_in[hd], 0);
        if (e != cudaSuccess) return cuda_fail(e, "host-to-device copy");
        aj_tensor t[8];
        const aj_tensor *ts[8];
        for (int i = 0; i < 8; ++i) {
            const bool is_q = i == 0 || i == 3 || i >= 6;
            const int64_t n = is_q ? pr.Nq : pr.Nk;
            t[i].ptr = (char *)(i < 6 ? p->d_in[i] : p->d_out[i - 6]) + hd * (is_q ? hq_bytes : hk_bytes);
            t[i].stride_n = pr.d; t[i].stride_h = n * pr.d; t[i].stride_b = n * pr.d;
            ts[i] = (no_tangents && ((i >= 3 && i <= 5) || i == 7)) ? nullptr : &t[i];
        }
        if (aj_status st = launch_schedule(p, p->head, 1, 1, ts, p->d_lse + (size_t)hd * pr.Nq, nullptr, stream, SLOT_HEAD + hd * SLOTS_PER_HEAD)) return st;
        e = cudaEventRecord(p->ev_k[hd], stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_out, p->ev_k[hd], 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync((char *)o + hd * hq_bytes, (char *)p->d_out[0] + hd * hq_bytes, hq_bytes, cudaMemcpyDeviceToHost, p->s_out);
        if (e == cudaSuccess && !no_tangents)
            e = cudaMemcpyAsync((char *)to + hd * hq_bytes, (char *)p->d_out[1] + hd * hq_bytes, hq_bytes, cudaMemcpyDeviceToHost, p->s_out);
        if (e == cudaSuccess && lse)
            e = cudaMemcpyAsync(lse + (size_t)hd * pr.Nq, p->d_lse + (size_t)hd * pr.Nq, pr.Nq * sizeof(float), cudaMemcpyDeviceToHost, p->s_out);
        if (e != cudaSuccess) return cuda_fail(e, "device-to-host copy");
    }
    e = cudaEventRecord(p->ev_end, p->s_out);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, p->ev_end, 0);
    if (e != cudaSuccess) return cuda_fail(e, "stream ordering");
    return AJ_OK;
}

aj_status attn_jvp_plan_tensor_map_stats(const aj_plan *p, int64_t *encodes, int64_t *hits) {
    if (!p) return fail(AJ_ERR_INVALID_ARG, "plan is NULL");
    std::lock_guard<std::mutex> lock(p->mu);
    if (encodes) *encodes = p->map_encodes;
    if (hits) *hits = p->map_hits;
    return AJ_OK;
}

}  // extern "C"
