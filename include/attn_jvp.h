/*
 * attn_jvp.h -- C ABI of the B200 (sm_100a) fused attention + JVP library.
 *
 * One pass over Q, K, V and their tangents tQ, tK, tV returns
 *     O   = softmax(mask(Q K^T * s)) V                         (Eq. 42)
 *     tO  = sum_b p_ab tV_b + sum_b p_ab (tS_ab - sum_c p_ac tS_ac) V_b   (Eq. 44)
 *     lse = log-sum-exp of the masked scaled scores             (Alg. 1 "L")
 * with tS = (tQ K^T + Q tK^T) * s (Eq. 43); masked entries have S = -inf and
 * tS = 0.  The computation is the online-softmax recurrence of PAPER.md:866-878
 * (Alg. 1) under the sparse query-group / key-range mask of PAPER.md:880-886.
 * Around that call: attn_fwd (the same without tangents, also for Nq != Nk), attn_bwd (the primal backward dQ, dK, dV
 * that consumes lse), attn_jvp_fwd_host (host buffers, copies pipelined head by head), and the host-only scheduler.
 *
 * Conventions
 *  - All functions are extern "C", never throw, never synchronise the stream (except plan creation / first-use
 *    schedule uploads and attn_jvp_plan_device_status, as stated there), and return an aj_status; attn_jvp_last_error() gives a thread-local message for the last failure.
 *  - The caller owns every tensor.  "device" pointers are CUDA device memory of the current
 *    device; "host" pointers are ordinary (preferably pinned) host memory.
 *  - Tensors are [B, H, N, d] with d contiguous; strides are in ELEMENTS (aj_tensor).
 *  - Supported: d in {64, 128}.  dtype AJ_BF16 runs tcgen05 / TMEM / TMA kernels: d = 128 on CTA pairs (the performance
 *    path, AJ_KERNEL_UMMA_PAIR), d = 64 on the single-CTA kernels (AJ_KERNEL_UMMA: forward, tangent-free forward and
 *    backward; the forward + JVP reaches about 0.6 of the bf16 tensor peak there and the backward about 0.3, against 0.9 and
 *    0.5 at d = 128).  AJ_FP32 (any supported d) runs the
 *    plain-FMA SIMT kernels (plain fp32 FMA for the 1e-4 tolerance, R14): a CORRECTNESS path two to three orders
 *    of magnitude slower (a few TFLOP/s), which attn_jvp_plan_kernel reports as AJ_KERNEL_SIMT.
 *    Anything else returns AJ_ERR_UNSUPPORTED.  There is no CPU fallback.
 *  - Inputs must be finite: masked-out tail keys are multiplied by an exact 0 (R15).
 *  - The CUDA device that is current when a plan is created owns the plan: every later call with that plan must be made
 *    with the same device current (else AJ_ERR_INVALID_ARG).  Plans of different devices may live in one process.
 *  - Input tensors may be broadcast over heads or batches with a zero stride on the SIMT kernels only (the tcgen05
 *    kernels return AJ_ERR_UNSUPPORTED); output tensors never (AJ_ERR_INVALID_ARG).
 *  - The enqueueing calls (attn_jvp_fwd, attn_jvp_fwd_tl, attn_fwd, and attn_bwd after its first call on a plan) make no
 *    allocation and no synchronisation: they can be captured into a CUDA graph.  The plan caches the TMA
 *    tensor maps it encodes per tensor argument and re-encodes one only when that argument's pointer or strides change.
 */
#ifndef ATTN_JVP_H_
#define ATTN_JVP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    AJ_OK = 0,
    AJ_ERR_INVALID_ARG = -1, /* null pointer, bad shape, misaligned pointer/stride, bad descriptor */
    AJ_ERR_UNSUPPORTED = -2, /* valid request this build has no kernel for (d, dtype)              */
    AJ_ERR_CUDA = -3,        /* a CUDA runtime/driver call failed (message has the CUDA error)     */
    AJ_ERR_OOM = -4          /* host or device allocation failed                                   */
} aj_status;

typedef enum { AJ_BF16 = 0, AJ_FP32 = 1 } aj_dtype;

/* Mask kinds (PAPER.md:175-180 Eq. 8 teacher forcing; :155 block-causal; :886 dense; :882-886 ranges). */
typedef enum {
    AJ_MASK_FULL = 0,            /* every query sees every key                                          */
    AJ_MASK_BLOCK_CAUSAL = 1,    /* block i sees blocks <= i                                             */
    AJ_MASK_TEACHER_FORCING = 2, /* packed [clean | noisy]: clean i -> clean <= i; noisy i -> clean < i
                                    and noisy i; nothing else                                             */
    AJ_MASK_RANGES = 3           /* explicit query groups with key-range lists                            */
} aj_mask_kind;

/* Structural zeros among the tangents: a PROMISE by the caller that lets the kernel skip contractions whose operand is
 * identically zero ("The tangent of the clean context is zero" in every TF-sCM call, and clean rows see
 * only clean keys, so their tangents stay zero in every layer).  The results are those of the dense computation on the
 * same data; data that breaks the promise gives undefined tO.
 *   DENSE      no promise (6 contractions per unmasked pair)
 *   CLEAN_ZERO TEACHER_FORCING: tQ, tK, tV rows of the clean half are zero -> clean x clean pairs need 2 of the 6
 *              contractions (S, P V), noisy x clean pairs 4 (no Q tK^T, no P tV), and tO of the clean rows is written as 0.
 *              RANGES: per-group / per-range flags (q_tangent_zero, k_tangent_zero) say the same.
 *   NONE       no tangents at all: plain masked attention forward (O, lse); tq, tk, tv, to may be NULL in attn_jvp_fwd
 *              (a non-NULL `to` is filled with zeros).  This is the cached-prefix forward of PAPER.md:324-328. */
typedef enum { AJ_TANGENT_DENSE = 0, AJ_TANGENT_CLEAN_ZERO = 1, AJ_TANGENT_NONE = 2 } aj_tangent_zero;

/* Kernel selection (attn_jvp_plan_set_kernel). AUTO = UMMA_PAIR when (bf16, d = 128), UMMA when (bf16, d = 64), else SIMT.
 * UMMA: one CTA per 128-row query tile (tcgen05.mma.cta_group::1).  UMMA_PAIR: a CTA pair per 256-row query tile
 * (tcgen05.mma.cta_group::2, M = 256; the two SMs share every K/V tile).
 * UMMA_PAIR sends the tasks that need no tangent at all (AJ_TASK_PRIMAL_ONLY: everything under AJ_TANGENT_NONE, the clean
 * rows under AJ_TANGENT_CLEAN_ZERO) to a second kernel specialised for them (two softmax warpgroups, S triple-buffered), in
 * a launch of its own before the general one; UMMA_PAIR_ONE keeps every task in the one general CTA-pair kernel. */
typedef enum { AJ_KERNEL_AUTO = 0, AJ_KERNEL_SIMT = 1, AJ_KERNEL_UMMA = 2, AJ_KERNEL_UMMA_PAIR = 3, AJ_KERNEL_UMMA_PAIR_ONE = 4 } aj_kernel;

/*
 * Mask descriptor = the paper's problem statement.  Structured kinds: a block is
 * chunk_frames * frame_len tokens (frame-wise c1-1: chunk_frames = 1; chunk-wise c3-3: 3;
 * PAPER.md:398); block 0 has first_chunk_frames frames if that is > 0.  num_frames counts latent
 * frames per half; the sequence must be num_frames*frame_len tokens (twice that for
 * TEACHER_FORCING, clean half first: PAPER.md:177).  AJ_MASK_RANGES: group g owns query rows
 * [q_begin[g], q_end[g]) and sees keys in the union of [k_begin[r], k_end[r]) for
 * r in [range_offset[g], range_offset[g+1]); groups must be disjoint, each group's ranges sorted
 * and disjoint, everything inside [0,Nq) x [0,Nk) (else AJ_ERR_INVALID_ARG).  The arrays are HOST
 * pointers and are copied by the call that receives the descriptor.  Rows in no group, or with an
 * empty key list, get O = 0, tO = 0, lse = -inf.
 */
typedef struct {
    int32_t kind;               /* aj_mask_kind */
    int32_t frame_len;          /* L tokens per latent frame */
    int32_t num_frames;         /* F frames (per half for TEACHER_FORCING) */
    int32_t chunk_frames;       /* frames per block */
    int32_t first_chunk_frames; /* 0 = same as chunk_frames */
    int32_t num_groups;         /* AJ_MASK_RANGES only, as are the arrays below */
    int32_t tangent_zero;       /* aj_tangent_zero */
    const int32_t *q_begin, *q_end, *range_offset, *k_begin, *k_end;
    /* AJ_MASK_RANGES with AJ_TANGENT_CLEAN_ZERO: non-zero = the tQ rows of group g / the tK, tV rows of range r are all
     * zero; [num_groups] / [range_offset[num_groups]]; NULL = no flag set.  Overlapping key ranges of different groups
     * must agree. */
    const int32_t *q_tangent_zero, *k_tangent_zero;
} aj_mask_desc;

typedef struct {
    int32_t B, H, Nq, Nk, d;
    int32_t dtype; /* aj_dtype of q,k,v,tq,tk,tv,o,to; lse is always fp32 */
    float scale;   /* softmax scale s applied to S and tS; 0 means 1/sqrt(d) */
} aj_problem;

/* A [B,H,N,d] tensor view: element strides, d contiguous. */
typedef struct {
    void *ptr;
    int64_t stride_b, stride_h, stride_n;
} aj_tensor;

/*
 * How query rows are cut into tiles.  PER_GROUP: tiles start at each query group's first row, so every row of a
 * tile sees the same keys ("i is a query tile inside Q_g").  PACKED: tiles lie on a global grid of
 * tile_q rows ("Split Q into query tiles"); a tile that straddles groups streams the union of
 * their key ranges and every entry carries the interval of tile rows that may see it (the other rows are masked,
 * PAPER.md:909-914).  Same results; PACKED wastes no rows at group ends.
 */
typedef enum { AJ_TILING_PER_GROUP = 0, AJ_TILING_PACKED = 1 } aj_tiling;

/* One unit of work: a query tile for one (b, h) ("tasks (g,i)").  Its keys are the schedule ENTRIES
 * [range_begin, range_begin + range_count): entry e = keys [k_begin[e], k_end[e]) seen by tile rows
 * [row_begin[e], row_end[e]) (relative to q_begin).  PER_GROUP: entries are the lowered key ranges (same indices as
 * attn_jvp_schedule_get) with rows [0, tile_q). */
typedef struct {
    int32_t b, h;
    int32_t q_begin, q_rows;          /* query rows [q_begin, q_begin + q_rows) */
    int32_t range_begin, range_count; /* its entries */
    int32_t num_kv_tiles;             /* key tiles it streams (sum over entries of ceil(len / tile_k)) */
    int32_t group;                    /* PER_GROUP: index of its query group; PACKED: -1 */
    int32_t flags;                    /* AJ_TASK_* */
} aj_task;

/* aj_task::flags.  PRIMAL_ONLY: tQ of every row and tK, tV of every key of the task are structurally zero: the task needs
 * only S = Q K^T and O += P V (tO = 0). */
enum { AJ_TASK_PRIMAL_ONLY = 1 };

typedef struct aj_schedule aj_schedule; /* host-only: groups, merged ranges, ordered task list */
typedef struct aj_plan aj_plan;         /* schedule + its device copy + staging buffers       */

/* ---- Host-side scheduler (no GPU needed): descriptor -> groups/ranges -> tile tasks (Alg. 1 input) ---- */

/* Lowers `mask` to disjoint query groups with sorted, merged key ranges, cuts every group into query
 * tiles of tile_q rows starting at the group start, and orders the tasks longest-first (ties: b, h,
 * group, tile).  tile_q, tile_k > 0.  *out is owned by the caller (attn_jvp_schedule_destroy). */
aj_status attn_jvp_schedule_create(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_q,
                                   int32_t tile_k, aj_schedule **out);
/* Same with an explicit aj_tiling (attn_jvp_schedule_create = AJ_TILING_PER_GROUP).  tile_q < 32768. */
aj_status attn_jvp_schedule_create_tiled(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_q,
                                         int32_t tile_k, int32_t tiling, aj_schedule **out);
/* The same mask seen from the KEYS (primal backward, dK and dV): "query groups" of the result are maximal key intervals
 * seen by the same rows, their "key ranges" are the sorted, merged query-row ranges that see them (keys no row sees
 * become range-less groups); tasks are tiles of tile_keys keys (per-group tiling) that stream their rows in tiles of
 * tile_rows.  attn_jvp_schedule_get / _info read it like any schedule, with the roles swapped. */
aj_status attn_jvp_schedule_create_transposed(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_keys,
                                              int32_t tile_rows, aj_schedule **out);
/* Same with an explicit aj_tiling of the KEY axis (PACKED: key tiles on a global grid of tile_keys keys; a tile that
 * straddles key intervals streams the union of their row ranges, each entry carrying the interval of tile keys it sees). */
aj_status attn_jvp_schedule_create_transposed_tiled(const aj_problem *problem, const aj_mask_desc *mask, int32_t tile_keys,
                                                    int32_t tile_rows, int32_t tiling, aj_schedule **out);
aj_status attn_jvp_schedule_destroy(aj_schedule *sched);
/* Any out pointer may be NULL. unmasked_pairs_per_head = sum over groups of rows * allowed keys. */
aj_status attn_jvp_schedule_info(const aj_schedule *sched, int32_t *num_groups, int32_t *num_ranges,
                                 int32_t *num_tasks, int64_t *unmasked_pairs_per_head);
/* Copy out the lowered mask: q_begin, q_end [num_groups]; range_offset [num_groups + 1];
 * k_begin, k_end [num_ranges]; tasks [num_tasks].  NULL pointers are skipped. */
aj_status attn_jvp_schedule_get(const aj_schedule *sched, int32_t *q_begin, int32_t *q_end,
                                int32_t *range_offset, int32_t *k_begin, int32_t *k_end, aj_task *tasks);

/* Copy out the entries the tasks index: k_begin, k_end, row_begin, row_end [num_entries].  NULL pointers are
 * skipped (call once with only num_entries to size the arrays). */
aj_status attn_jvp_schedule_entries(const aj_schedule *sched, int32_t *num_entries, int32_t *k_begin,
                                    int32_t *k_end, int32_t *row_begin, int32_t *row_end);

/* Per entry: non-zero = the tK, tV rows of its keys are structurally zero (aj_tangent_zero).  [num_entries]. */
aj_status attn_jvp_schedule_entry_flags(const aj_schedule *sched, int32_t *key_tangent_zero);
/* Unmasked pairs per head by the number of contractions they need: pairs[0] need 2 (tQ row and tK, tV key zero),
 * pairs[1] need 4 (only the key's tangents zero), pairs[2] need all 6.  Sums to unmasked_pairs_per_head. */
aj_status attn_jvp_schedule_pair_classes(const aj_schedule *sched, int64_t pairs[3]);

/* Static assignment of the tasks to num_workers persistent workers (the CTA-pair kernel's SM pairs; PAPER.md:897
 * "parallel over tasks"): tasks are taken (b, h)-major, longest first inside a head, and each goes to the worker that
 * is free first under a cost model (a constant per task plus, per pair of key tiles, a weight that depends on how many
 * contractions the pair needs).  worker_offset [num_workers + 1], task_ids
 * [num_tasks] (indices into the task list of attn_jvp_schedule_get): worker w runs
 * task_ids[worker_offset[w] .. worker_offset[w+1]) in order.  Every task appears exactly once. */
aj_status attn_jvp_schedule_assign(const aj_schedule *sched, int32_t num_workers, int32_t *worker_offset,
                                   int32_t *task_ids);

/* ---- Plans and the forward call ---- */

/* Validates the problem, builds the schedule for the kernel that will run and uploads it (one H2D copy,
 * synchronous).  Needs a CUDA device.  Errors: INVALID_ARG, UNSUPPORTED, CUDA, OOM. */
aj_status attn_jvp_plan_create(const aj_problem *problem, const aj_mask_desc *mask, aj_plan **out);
aj_status attn_jvp_plan_destroy(aj_plan *plan);
aj_status attn_jvp_plan_info(const aj_plan *plan, int64_t *unmasked_pairs_per_head, int32_t *num_tasks);
/* attn_jvp_schedule_pair_classes of the plan's mask. */
aj_status attn_jvp_plan_pair_classes(const aj_plan *plan, int64_t pairs[3]);
/* Force a kernel (debugging / comparison).  Rebuilds and re-uploads the schedule.  A kernel on a problem it does not
 * cover (a tcgen05 kernel on fp32 inputs, a CTA-pair kernel on d = 64) returns AJ_ERR_UNSUPPORTED and leaves the plan
 * unchanged. */
aj_status attn_jvp_plan_set_kernel(aj_plan *plan, int32_t kernel);
/* Force a query tiling (aj_tiling).  Default: PACKED for the tcgen05 kernels, PER_GROUP for the SIMT kernel; the SIMT
 * kernel supports only PER_GROUP and the CTA-pair kernel only PACKED (AJ_ERR_UNSUPPORTED otherwise).  Rebuilds and re-uploads the schedule; results do not change. */
aj_status attn_jvp_plan_set_tiling(aj_plan *plan, int32_t tiling);
/*
 * Rendezvous of the CTA-pair forward kernel's workers (AJ_KERNEL_UMMA_PAIR / _ONE).  On long sequences every SM pair streams
 * the keys of its task on its own schedule; the pairs drift apart and each ends up reading K, tK, V, tV from DRAM instead of
 * sharing them through L2 (N = 115,200, 24 heads, full mask: 379 GB read per launch for 5.7 GB of inputs).  With a rendezvous
 * the producers of all pairs meet -- at every task slot of their lists (PER_SLOT: for schedules whose tasks cost the same), or
 * whenever they enter a new head (PER_HEAD: tasks of different cost; the lists are then levelled at every head) -- through
 * plan-owned counters that a cudaMemsetAsync on the call's stream clears before every launch.  The wait is bounded (a pair
 * that waits in vain three times stops waiting for the rest of the launch): a performance hint, never a correctness condition;
 * results are bit-identical in every mode.
 *   AUTO      (default) the library turns a mode on where it pays: the longest key stream of a task exceeds what L2 keeps for
 *             all pairs (48 MB) and the schedule has the shape the mode needs.
 *   OFF / PER_SLOT / PER_HEAD  force it.  PER_SLOT is ignored on plans with primal-only task lists (AJ_TANGENT_CLEAN_ZERO);
 *             both are ignored by kernels other than the CTA-pair forward.  attn_jvp_plan_rendezvous reports what is in effect.
 * Rebuilds and re-uploads the forward schedule (synchronous).  ONE LAUNCH AT A TIME while a mode is in effect: two launches of
 * the same plan that overlap on the GPU (two streams) share the counters -- the second launch's memset clears what the first
 * is counting -- so pairs wait for their time-outs (up to 3 x 1.5 M clk each) and the L2 sharing is lost.  Results stay
 * right.  Callers that overlap launches of one plan should set OFF or use one plan per stream.
 */
typedef enum { AJ_RENDEZVOUS_AUTO = 0, AJ_RENDEZVOUS_OFF = 1, AJ_RENDEZVOUS_PER_SLOT = 2, AJ_RENDEZVOUS_PER_HEAD = 3 } aj_rendezvous;
aj_status attn_jvp_plan_set_rendezvous(aj_plan *plan, int32_t mode);
/* *in_effect = AJ_RENDEZVOUS_OFF, PER_SLOT or PER_HEAD: what attn_jvp_fwd on this plan does now. */
aj_status attn_jvp_plan_rendezvous(const aj_plan *plan, int32_t *in_effect);
/*
 * Worker budget of the CTA-pair kernels (forward, forward-only, backward): they are persistent, one CTA pair per SM pair
 * with a host-assigned task list each, and by default take every pair of the device (74 on a B200).  A caller that runs
 * something else beside them -- the NCCL kernels of the Ulysses all-to-all of the next head group, a
 * copy kernel -- can leave it room: num_pairs > 0 builds the lists for that many pairs (the grid and the rendezvous targets
 * follow), 0 restores the default.  Without a budget a pair whose SMs are held by another kernel starts its whole list
 * late, and the launch ends when that pair does.  Results do not depend on the budget.  Rebuilds and re-uploads the forward
 * schedule (synchronous); the backward schedules are rebuilt on the next attn_bwd.  Ignored by the single-CTA and SIMT kernels.
 */
aj_status attn_jvp_plan_set_workers(aj_plan *plan, int32_t num_pairs);
/* How many CTA pairs attn_jvp_fwd launches for the general kernel and for the forward-only kernel of the primal-only tasks
 * (either pointer may be NULL; 0 when that kernel is not launched). */
aj_status attn_jvp_plan_workers(const aj_plan *plan, int32_t *num_pairs, int32_t *num_primal_pairs);
/* Which kernel attn_jvp_fwd will launch (aj_kernel, never AUTO) and how many kernel launches one
 * attn_jvp_fwd call makes. */
aj_status attn_jvp_plan_kernel(const aj_plan *plan, int32_t *kernel, int32_t *launches_per_call);

/*
 * Enqueues the fused forward + JVP on `cuda_stream` (a cudaStream_t; NULL = default stream) and returns
 * without waiting.  q, tq: [B,H,Nq,d]; k, v, tk, tv: [B,H,Nk,d]; o, to: [B,H,Nq,d] in the problem dtype;
 * lse: contiguous fp32 [B,H,Nq] (may be NULL).  All DEVICE memory; inputs are only read.  Pointers must be
 * 16-byte aligned and strides multiples of 8 elements, stride_n >= d (else AJ_ERR_INVALID_ARG).
 * The forward calls keep no per-call device state in the plan, except the rendezvous counters of long-sequence plans
 * (attn_jvp_plan_set_rendezvous: one launch at a time while a mode is in effect): otherwise one plan may be enqueued on several
 * streams at the same time (the tensor-map cache is guarded by a mutex).  attn_bwd and the host-buffer calls own a workspace /
 * staging buffers in the plan: one such call at a time per plan.
 * Plans whose mask says AJ_TANGENT_NONE never read tq, tk, tv (they may be NULL), fill a non-NULL `to` with zeros and
 * write O and lse only -- on every kernel (CTA-pair and single-CTA tcgen05, SIMT).
 */
aj_status attn_jvp_fwd(const aj_plan *plan, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v,
                       const aj_tensor *tq, const aj_tensor *tk, const aj_tensor *tv, const aj_tensor *o,
                       const aj_tensor *to, float *lse, void *cuda_stream);

/* attn_jvp_fwd that also returns the tangent of lse along the input tangents,
 *     tlse_a = sum_b p_ab tS_ab = r_a / l_a        (r is the running sum the recurrence carries anyway)
 * i.e. d/d eps of log sum_b exp(S_ab + eps tS_ab), which a layer-level JVP that consumes L needs.
 * tlse: contiguous fp32 [B,H,Nq], DEVICE memory, or NULL (then identical to attn_jvp_fwd).  0 for rows without keys,
 * for rows whose tangents are structurally zero, and on AJ_TANGENT_NONE plans. */
aj_status attn_jvp_fwd_tl(const aj_plan *plan, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v,
                          const aj_tensor *tq, const aj_tensor *tk, const aj_tensor *tv, const aj_tensor *o,
                          const aj_tensor *to, float *lse, float *tlse, void *cuda_stream);

/* Masked attention forward without tangents: attn_jvp_fwd(plan, q, k, v, NULL, NULL, NULL, o, NULL, lse, stream) on a plan
 * whose mask says AJ_TANGENT_NONE (else AJ_ERR_INVALID_ARG).  q: [B,H,Nq,d], k, v: [B,H,Nk,d] (Nq != Nk allowed: the
 * current chunk against the cached prefix). */
aj_status attn_fwd(const aj_plan *plan, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v, const aj_tensor *o,
                   float *lse, void *cuda_stream);

/*
 * Primal backward under the plan's mask (Eq. 19: the student's gradient flows through
 * the ordinary primal path, for which the forward returns L): the vector-Jacobian product of Eq. 42,
 *     dV_b = sum_a p_ab dO_a,  dS_ab = p_ab (<dO_a, v_b> - <dO_a, O_a>),  dQ_a = s sum_b dS_ab k_b,  dK_b = s sum_a dS_ab q_a
 * with p_ab = exp(s <q_a, k_b> - lse_a) over the unmasked pairs.  q, o, dout, dq: [B,H,Nq,d]; k, v, dk, dv: [B,H,Nk,d]
 * in the problem dtype; lse: contiguous fp32 [B,H,Nq] as written by attn_jvp_fwd / attn_fwd on the same q, k, v.  All
 * DEVICE memory, same alignment rules as attn_jvp_fwd.  Every element of dq, dk, dv is written (0 for rows without
 * keys and keys no row sees).  Enqueues three kernels on `cuda_stream` (delta = <dO, O>; a pass with query tiles
 * stationary for dQ; a pass with key tiles stationary, on the transposed schedule, for dK and dV -- no atomics); the
 * first call on a plan also builds and uploads the two backward schedules (synchronous host work) and allocates a
 * [B,H,Nq] fp32 workspace.  bf16: tcgen05 / TMEM / TMA kernels (bf16 P and dS operands, fp32 accumulation; d = 128 on CTA
 * pairs, d = 64 and plans forced to AJ_KERNEL_UMMA on single CTAs); fp32 inputs, or a plan forced to AJ_KERNEL_SIMT: plain
 * fp32 FMA kernels.
 */
aj_status attn_bwd(aj_plan *plan, const aj_tensor *q, const aj_tensor *k, const aj_tensor *v, const aj_tensor *o,
                   const float *lse, const aj_tensor *dout, const aj_tensor *dq, const aj_tensor *dk, const aj_tensor *dv,
                   void *cuda_stream);

/*
 * Same computation on HOST buffers: contiguous [B,H,N,d] arrays in the problem dtype (lse fp32
 * [B,H,Nq], may be NULL).  Copies the six inputs to plan-owned device staging buffers (allocated on
 * first use), runs attn_jvp_fwd, copies o, to, lse back, all asynchronously on `cuda_stream`; the
 * caller synchronises the stream before reading the outputs.  Pinned host memory is needed for the
 * copies to overlap; pageable memory works but is staged by the runtime.  The heads are processed one by one (copy-in,
 * kernel and copy-out of neighbouring heads overlap on three streams).  AJ_TANGENT_NONE plans accept tq = tk = tv = to =
 * NULL (all four): only q, k, v go up and o, lse come back.
 */
aj_status attn_jvp_fwd_host(aj_plan *plan, const void *q, const void *k, const void *v, const void *tq,
                            const void *tk, const void *tv, void *o, void *to, float *lse,
                            void *cuda_stream);

/*
 * attn_bwd on HOST buffers (SURVEY.md 8(b) conventions as attn_jvp_fwd_host): contiguous [B,H,N,d] arrays in the problem
 * dtype, lse contiguous fp32 [B,H,Nq].  Head by head: q, k, v, o, dout, lse go up on a copy-in stream, the head's three
 * kernels run on `cuda_stream` as soon as they have landed, dq, dk, dv come back on a copy-out stream; `cuda_stream`
 * finally waits for the last copy.  The caller synchronises the stream before reading the outputs.  Staging buffers,
 * per-head schedules, copy streams and events are plan-owned and created on first use.
 */
aj_status attn_bwd_host(aj_plan *plan, const void *q, const void *k, const void *v, const void *o, const float *lse,
                        const void *dout, void *dq, void *dk, void *dv, void *cuda_stream);

/*
 * attn_bwd for callers that cannot allocate device memory: no plan, no cudaMalloc / cudaFree, no allocating library call, on
 * the first call or any later one.  It exists for host programs in which a library-side allocation is not an option -- a
 * process whose own memory pool claimed the GPU at start-up (a raw cudaMalloc then fails, or takes memory the pool counts as
 * its own), and step loops with a latency budget, where an allocation can hold up every stream of the device.  Such a caller
 * could not even create a plan, so the mask is passed as its descriptor and evaluated inside the kernels.
 *
 * Computes exactly what attn_bwd computes (PAPER.md:247 Eq. 19, :945), with the plain-FMA fp32 kernels (both dtypes, d in
 * {64, 128}; a few TFLOP/s: a correctness-grade path, not the tcgen05 one).  problem / mask as for attn_jvp_plan_create; mask
 * kinds FULL (Nq != Nk allowed), BLOCK_CAUSAL and TEACHER_FORCING; AJ_MASK_RANGES returns AJ_ERR_UNSUPPORTED (its lists would
 * need device memory), and the mask's tangent_zero field is ignored (the backward has no tangents).  Tensors, lse, alignment
 * rules and `cuda_stream` as for attn_bwd; all DEVICE memory of the current device, owned by the caller; every element of
 * dq, dk, dv is written.  Enqueues three kernels and returns without waiting.
 *
 * Scratch.  The one intermediate, delta_a = <dO_a, O_a> per query row, lives in a fixed array inside the library's device
 * image: AJ_STATIC_SCRATCH_MAX_ROWS floats (4 MiB) on every GPU that loads the library, held until the process exits.
 *  - Limit: B * H * Nq <= AJ_STATIC_SCRATCH_MAX_ROWS, else AJ_ERR_INVALID_ARG with a message that names both numbers
 *    (BASELINE.json's config 2, 12 heads x 65,520 rows, fits; larger launches go head group by head group).
 *  - Every call on a device uses the SAME array.  Each call writes the rows it will read before reading them, so nothing has
 *    to be cleared between calls and stale contents are harmless; but two calls that can overlap on the GPU (different
 *    streams, or different host threads without ordering between their streams) race on it and give wrong gradients.
 *    Calls on one stream, or on streams ordered by events, are safe.
 *  - The first call made with a given device current looks up the array's address on that device and raises the kernels'
 *    shared-memory limit (no allocation, but possibly the lazy load of the device image): make that first call ahead of
 *    time, outside any stream capture.  Later calls on that device only check arguments and launch.
 */
#define AJ_STATIC_SCRATCH_MAX_ROWS 1048576
aj_status attn_bwd_static(const aj_problem *problem, const aj_mask_desc *mask, const aj_tensor *q, const aj_tensor *k,
                          const aj_tensor *v, const aj_tensor *o, const float *lse, const aj_tensor *dout,
                          const aj_tensor *dq, const aj_tensor *dk, const aj_tensor *dv, void *cuda_stream);

/* How many TMA tensor maps the plan has encoded so far and how many calls found theirs in the plan's cache (either
 * pointer may be NULL).  Steady-state calls on unchanged tensors encode nothing. */
aj_status attn_jvp_plan_tensor_map_stats(const aj_plan *plan, int64_t *encodes, int64_t *hits);

/*
 * Device-side health of the plan's last launches: synchronises the device, then *code = 0 if every
 * attn_jvp_fwd on this plan ran to completion, else a non-zero internal code (a pipeline wait of the
 * tcgen05 kernel timed out and the launch was abandoned: its outputs are garbage).  Resets the code.
 * Returns AJ_ERR_CUDA if the device itself reports an error.
 */
aj_status attn_jvp_plan_device_status(aj_plan *plan, int32_t *code);

/* Message for the most recent non-OK status returned to this thread ("" if none). Never NULL. */
const char *attn_jvp_last_error(void);
/* Library version string, e.g. "attn_jvp 0.2 (sm_100a)". */
const char *attn_jvp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ATTN_JVP_H_ */
