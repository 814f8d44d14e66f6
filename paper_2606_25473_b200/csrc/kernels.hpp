// Kernel launch interfaces (internal).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>

#include "attn_jvp.h"

namespace aj {

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the (kernel, device) pair: `done` is one bit per device ordinal
// of a kernel's launcher (ordinals >= 64 set the attribute on every launch).  Safe from several host threads.
template <typename K>
inline cudaError_t ensure_dynamic_smem(K *kernel, int bytes, std::atomic<uint64_t> &done) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint64_t bit = dev < 64 ? (1ull << dev) : 0ull;
    if (bit && (done.load(std::memory_order_acquire) & bit)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && bit) done.fetch_or(bit, std::memory_order_release);
    return e;
}

constexpr int SIMT_TILE_Q = 16;
constexpr int SIMT_TILE_K = 32;
constexpr int UMMA_TILE_Q = 128;  // B_r: query rows per task = UMMA M
constexpr int UMMA_TILE_K = 64;   // B_c: keys per streamed tile
constexpr int UMMA_PAIR_TILE_Q = 256;  // query rows per task of the CTA-pair kernel (UMMA M = 256 over two SMs)

struct SimtParams {
    aj_tensor q, k, v, tq, tk, tv, o, to;   // no_tangents: tq, tk, tv are never read; to.ptr may be NULL
    float *lse;
    float *tlse;                            // [B, H, Nq] tangent of lse (r / l) or NULL
    int32_t no_tangents;                    // AJ_TANGENT_NONE plans: plain masked attention, tO = 0, tlse = 0
    const aj_task *tasks;
    const int32_t *k_begin, *k_end;
    int32_t H, Nq;
    float scale;
};

cudaError_t launch_simt(const SimtParams &prm, int dtype, int d, int num_tasks, cudaStream_t stream);

// Primal backward, plain FMA (kernel_simt_bwd.cu): a delta kernel, a dQ kernel over q_tasks and a dK/dV kernel over
// k_tasks (the transposed schedule: key tiles with the row ranges that see them)
struct BwdParams {
    aj_tensor q, k, v, o, dout, dq, dk, dv;
    const float *lse;                 // [B, H, Nq] from the forward
    float *delta;                     // [B, H, Nq] workspace: <dO_a, O_a> (may be NULL when `ld` is given)
    float2 *ld;                       // [B, H, Nq] workspace of the CTA-pair kernels: {lse * log2(e), delta} (or NULL)
    uint4 *aug;                       // [2][B, H, Nq] rows of 32 B = 2 x uint4: the 16 extra K columns -lse/s and -delta (or NULL)
    const aj_task *q_tasks; const int32_t *q_kb, *q_ke;   // query tiles and their key ranges
    const aj_task *k_tasks; const int32_t *k_rb, *k_re;   // key tiles and their row ranges
    int32_t B, H, Nq;
    float scale;
};
cudaError_t launch_bwd_simt(const BwdParams &prm, int dtype, int d, int num_q_tasks, int num_k_tasks, cudaStream_t stream);

// Primal backward on tcgen05 (kernel_umma_bwd_sm100.cu; bf16, d = 128 or 64): one pass with query tiles stationary (dQ),
// one with key tiles stationary (dK, dV).  a1, a2: stationary operands (box {64, 128}); b1, b2: streamed (box {64, 64}).
struct BwdUmmaParams {
    CUtensorMap tm_a1, tm_a2, tm_b1, tm_b2;
    aj_tensor out1, out2;             // dQ | dK, dV
    aj_tensor a1, a2;                 // dQ pass: Q and dO again as plain views (their rows go to TMEM, not to shared memory)
    int32_t Na;                       // rows of the stationary tensors
    const float *lse, *delta;         // [B, H, Nq]
    const aj_task *tasks;
    const int32_t *r_begin, *r_end;   // the tasks' streamed ranges
    const int32_t *cta_off, *cta_ids; // CTA c runs tasks cta_ids[cta_off[c] .. cta_off[c+1]) (head-major, host-assigned)
    int32_t *err;                     // abort code word of the plan
    int32_t num_tasks, H, Nq;
    float scale, scale_log2;
};
cudaError_t launch_bwd_umma(const BwdUmmaParams &prm, int d, bool keys, int grid, cudaStream_t stream);

// Primal backward on CTA pairs (kernel_umma_bwd_pair_sm100.cu; bf16, d = 128): tcgen05.mma.cta_group::2, 256 stationary rows
// per pair, packed tiling (entries carry row intervals).  a1, a2: stationary operands (box {64, 128}; KEYS pass only);
// b1, b2: streamed (box {64, 64}); aug1, aug2: 2-D maps over the augmentation rows (16 bf16 each) of -lse/s and -delta, box
// {16, 64} (KEYS pass).
struct BwdPairParams {
    CUtensorMap tm_a1, tm_a2, tm_b1, tm_b2, tm_aug1, tm_aug2;
    CUtensorMap tm_b1h, tm_b2h;       // dQ pass, tile ping-pong form: streamed operands with box {64, 32} (half a tile per CTA)
    aj_tensor out1, out2;             // dQ | dK, dV
    aj_tensor a1, a2;                 // dQ pass: Q and dO as plain views (their rows go to TMEM, not to shared memory)
    const float2 *ld;                 // [B, H, Nq] {lse log2e, delta}
    const aj_task *tasks;
    const int32_t *r_begin, *r_end;   // schedule entries: streamed rows [r_begin[e], r_end[e]) ...
    const uint32_t *rows;             // ... seen by stationary tile rows [rows[e] & 0xffff, (rows[e] >> 16) & 0x7fff)
    const int32_t *pair_off, *pair_ids;
    int32_t *err;                     // abort code word of the plan
    int32_t num_tasks, H, Nq;
    float scale, scale_log2;
};
cudaError_t launch_bwd_umma_pair(const BwdPairParams &prm, bool keys, int num_pairs, cudaStream_t stream);
// delta kernel of kernel_simt_bwd.cu alone (shared by both backward paths)
cudaError_t launch_bwd_delta(const BwdParams &prm, int dtype, int d, cudaStream_t stream);

// bf16, d = 128 or 64, tcgen05 + TMEM + TMA (kernel_umma_sm100.cu; the CTA-pair kernels below take d = 128 only)
struct UmmaParams {
    CUtensorMap tm_q, tm_tq;    // box {64, 128, 1, 1} over [B, H, Nq, d], SWIZZLE_128B
    CUtensorMap tm_k, tm_tk, tm_v, tm_tv;  // box {64, 64, 1, 1} over [B, H, Nk, d], SWIZZLE_128B
    aj_tensor o, to;
    float *lse;
    float *tlse;                // [B, H, Nq] tangent of lse (r / l) or NULL
    const aj_task *tasks;
    const int32_t *k_begin, *k_end;   // schedule entries: keys [k_begin[e], k_end[e]) ...
    const uint32_t *rows;             // ... seen by tile rows [rows[e] & 0xffff, rows[e] >> 16)
    int32_t *counters;          // [2] abort code ([0], [1] unused)
    const int32_t *pair_off, *pair_ids;   // worker w (an SM pair; an SM of the single-CTA kernel) runs tasks pair_ids[pair_off[w] .. pair_off[w+1])
    // CTA-pair forward kernel, uniform-cost schedules whose per-head key stream does not fit in L2 (full masks of long sequences):
    // pair w enters the i-th task of its list only when slot_sync[i] has reached slot_expect[i] (all pairs that have an i-th task
    // have arrived), so that the pairs keep streaming the same keys at the same time; NULL = off.  Zeroed before every launch.
    int32_t *slot_sync;
    const int32_t *slot_expect;
    int32_t sync_per_head;      // 0: the counters are per task slot; 1: per (b, h), and the pairs meet when they enter a new head
    int32_t num_tasks, H, Nq;
    float scale_log2;           // s * log2(e)
    float scale;                // s
};

size_t umma_smem_bytes();
// primal: AJ_TANGENT_NONE plans (tq, tk, tv maps unused; tO = 0, tlse = 0)
cudaError_t launch_umma(const UmmaParams &prm, int d, bool primal, int grid, cudaStream_t stream);

// bf16, d = 128, CTA pairs: tcgen05.mma.cta_group::2 with M = 256 (kernel_umma_pair_sm100.cu)
size_t umma_pair_smem_bytes();
cudaError_t launch_umma_pair(const UmmaParams &prm, int num_pairs, cudaStream_t stream);

// bf16, d = 128, CTA pairs, primal-only tasks alone (no tangents: S and P~ V): two softmax warpgroups on alternate pair-steps,
// S triple-buffered in TMEM (kernel_umma_pair_fwd_sm100.cu).  prm.pair_off / pair_ids must list primal-only tasks only.
cudaError_t launch_umma_pair_fwd(const UmmaParams &prm, int num_pairs, cudaStream_t stream);

}  // namespace aj
