// bf16 attention + JVP for sm_100a: TMA -> shared-memory ring -> tcgen05.mma with TMEM accumulators.
//
// What it computes: Algorithm 1 of the paper for one task = one 128-row query tile of one
// query group, streaming the group's key ranges in 64-key tiles:
//   S  = Q K^T, tS = tQ K^T + Q tK^T            (Eq. 42-43; 3 MMAs, fp32 accumulators in TMEM)
//   P~ = exp2((S - m_ref) * s*log2e), H~ = P~ o (s * tS), l += rowsum P~, r += rowsum H~
//   O += P~ V,  T += P~ tV + H~ V                (3 MMAs, A operand = bf16 P~/H~ read from TMEM)
//   epilogue: O/l, lse = ln2 * (m_ref + log2 l), tO = T/l - (r/l)(O/l)          (Eq. 45)
// What differs from the paper's kernel: A and B of PAPER.md:872 are one accumulator
// T (both get the same rescale and are only ever summed); the reference max m_ref is only moved when the tile
// max exceeds it by 2^8 (lazy rescale; P~ <= 256), which leaves Eq. 45 unchanged; exp is base 2.
//
// CTA = 8 warps, persistent, one CTA per SM, each with its own host-assigned task list (head-major: assign_workers):
//   warp 0      TMA producer (one lane): next task of the list, Q/tQ tile, ring of {K,tK} / {V,tV} half-stages
//   warp 1      MMA issuer (whole warp runs the loop so every descriptor stays in uniform registers, one elected
//               lane issues): QK(j+1) is issued before PV(j) so the tensor pipe never waits on softmax
//   warp 2      TMEM allocator
//   warps 4-7   softmax + tangent weights + lazy rescale + epilogue; thread = one query row (TMEM lane)
// TMEM columns (fp32): O [0,128) | T [128,256) | S0 [256,320) tS0 [320,384) | S1 [384,448) tS1 [448,512);
// P~ and H~ (bf16, 32 columns each) overwrite the first half of their S / tS buffer.
// The six contractions of a tile are four MMA shapes (operands adjacent in shared memory / TMEM):
//   [S | tS]  = Q [K ; tK]^T   (N = 128)      tS += tQ K^T      (N = 64)       -- 2 x 8 instructions (K = 16 each)
//   [O | T]  += P~ [V | tV]    (N = 256)      T  += H~ V        (N = 128)      -- 2 x 4 instructions
// which cuts the operand bytes read from shared memory per tile from 192 KB to 160 KB (the 128 B/clk shared-memory
// port, not the tensor pipe, bounds the N = 64 shapes) and the issue count from 36 to 24.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

#include "kernels.hpp"
#include "umma_ptx.cuh"

namespace aj {

namespace {

constexpr int BR = UMMA_TILE_Q;        // 128 query rows
constexpr int BC = UMMA_TILE_K;        // 64 keys per tile
constexpr uint32_t QHALF_BYTES = BR * 64 * 2;      // one 64-column swizzle block of Q: 16 KB
constexpr uint32_t KVHALF_BYTES = BC * 64 * 2;     // one 64-column swizzle block of a streamed tile: 8 KB
// Head dimension D = 128 (two 64-column swizzle blocks per operand row) or 64 (one): the same kernel, with the K loops, the
// accumulator widths and the slot layouts following D.
template <int D> struct Cfg {
    static_assert(D == 64 || D == 128, "d must be 64 or 128");
    static constexpr int NSTAGE = D == 128 ? 5 : 10;                    // ring slots ({K,tK} or {V,tV} of one tile)
    static constexpr uint32_t Q_BYTES = BR * D * 2;                      // 32 KB | 16 KB
    static constexpr uint32_t KV_BYTES = BC * D * 2;                     // 16 KB | 8 KB
    static constexpr uint32_t SLOT_BYTES = 2 * KV_BYTES;                 // 32 KB | 16 KB
    static constexpr uint32_t SMEM_TILES = 2 * Q_BYTES + NSTAGE * SLOT_BYTES;   // 224 KB | 192 KB
    static constexpr uint32_t SMEM_TOTAL = SMEM_TILES + 1024 /*align*/ + 256 /*barriers*/;
    static constexpr uint32_t TM_T = D;                                  // O [0, D) | T [D, 2 D)
};
constexpr int MAX_STAGE = 10;
constexpr int NTHREADS = 256;

constexpr uint32_t TM_O = 0, TM_S0 = 256, TM_TS0 = 320, TM_SBUF = 128;  // S1 = S0 + 128, ...
constexpr float RESCALE_THRESHOLD = 8.0f;  // log2 units
constexpr float M_UNSET = -1.0e30f;        // reference max of a row that has not met an unmasked key yet (finite on purpose)

// Barrier indices inside the shared barrier array.
enum {
    BAR_Q_FULL = 0, BAR_Q_EMPTY,
    BAR_KV_FULL, BAR_KV_EMPTY = BAR_KV_FULL + MAX_STAGE,
    BAR_S_FULL = BAR_KV_EMPTY + MAX_STAGE, BAR_P_FULL = BAR_S_FULL + 2, BAR_H_FULL = BAR_P_FULL + 2, BAR_PV_DONE = BAR_H_FULL + 2,
    BAR_TASK_FULL = BAR_PV_DONE + 2, BAR_TASK_EMPTY = BAR_TASK_FULL + 2, NUM_BARS = BAR_TASK_EMPTY + 2
};

using namespace ptx;

// Instruction descriptor for kind::f16: D fp32 (bits 4-5 = 1), A and B bf16 (bits 7-9, 10-12 = 1), B major (bit 16),
// N >> 3 (bits 17-22), M >> 4 (bits 24-28).
__host__ __device__ constexpr uint32_t make_idesc(int n, bool b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(BR >> 4) << 24);
}
constexpr uint32_t IDESC_QK2 = make_idesc(2 * BC, false);  // 128 x 128 x 16: [S | tS] = Q [K ; tK]^T, A and B K-major
constexpr uint32_t IDESC_QK1 = make_idesc(BC, false);      // 128 x  64 x 16: tS += tQ K^T
// [O | T] += P~ [V | tV] is 128 x 2 D x 16 and T += H~ V is 128 x D x 16 (A from TMEM, B MN-major): make_idesc(2 * D | D, true)
constexpr uint32_t DESC_HI = desc_hi(1024);                // 8-row (K-major) / 8-key (MN-major) groups are 1024 B apart
constexpr uint32_t LBO_K = desc_lo_lbo(16);                // K-major with 128 B swizzle: unused, canonical value
constexpr uint32_t LBO_V = desc_lo_lbo(KVHALF_BYTES);      // MN-major: 64-column blocks [V h0 | V h1 | tV h0 | tV h1] 8 KB apart

// Walks the key tiles of a task in order: schedule entries [rb, rb + rc), each cut into BC-key tiles from its start.
struct TileCursor {
    const int32_t *kb, *ke;
    int r, rend, k, kend;
    __device__ void init(const int32_t *k_begin, const int32_t *k_end, int rb, int rc) {
        kb = k_begin; ke = k_end; r = rb; rend = rb + rc;
        if (r < rend) { k = kb[r]; kend = ke[r]; } else { k = 0; kend = 0; }
    }
    __device__ int key_row() const { return k; }
    __device__ int valid() const { return min(BC, kend - k); }
    __device__ int entry() const { return r; }
    __device__ void next() {
        k += BC;
        if (k >= kend) { ++r; if (r < rend) { k = kb[r]; kend = ke[r]; } }
    }
};

struct Shared {
    uint64_t bars[NUM_BARS];
    uint32_t tmem_base;
    int task_id[2];
    int abort_flag;
};

// PRIMAL: AJ_TANGENT_NONE plans -- plain masked attention (S and P~ V only): tQ, tK, tV are never loaded, the tS / T columns
// and the H~ hand-over are unused, tO = 0 and tlse = 0 are written where the caller gave the pointers.
template <int D, bool PRIMAL>
__global__ void __launch_bounds__(NTHREADS, 1)
attn_jvp_umma_kernel(const __grid_constant__ UmmaParams prm) {
    using C = Cfg<D>;
    constexpr int NSTAGE = C::NSTAGE;
    constexpr uint32_t Q_BYTES = C::Q_BYTES, SLOT_BYTES = C::SLOT_BYTES, SMEM_TILES = C::SMEM_TILES, TM_T = C::TM_T;
    constexpr uint32_t IDESC_PV2 = make_idesc(2 * D, true), IDESC_PV1 = make_idesc(D, true);
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;       // 1024-byte alignment for the 128-byte swizzle
    Shared *sh = reinterpret_cast<Shared *>(smem_raw + (tiles - raw) + SMEM_TILES);
    const uint32_t sQ = tiles, sTQ = tiles + Q_BYTES, sRing = tiles + 2 * Q_BYTES;
    const uint32_t bars = smem_u32(sh->bars);
    const Waiter wait{bars, &sh->abort_flag, prm.counters + 2};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * BAR_Q_FULL, 1);
        mbar_init(bars + 8 * BAR_Q_EMPTY, 1);
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bars + 8 * (BAR_KV_FULL + i), 1); mbar_init(bars + 8 * (BAR_KV_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bars + 8 * (BAR_S_FULL + i), 1);
            mbar_init(bars + 8 * (BAR_P_FULL + i), 128);
            mbar_init(bars + 8 * (BAR_H_FULL + i), 128);
            mbar_init(bars + 8 * (BAR_PV_DONE + i), 1);
            mbar_init(bars + 8 * (BAR_TASK_FULL + i), 1);
            mbar_init(bars + 8 * (BAR_TASK_EMPTY + i), 5);   // MMA warp + one lane of each softmax warp
        }
        sh->abort_flag = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sh->tmem_base)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sh->tmem_base;

    if (warp == 0) {
        // ================================================= TMA producer ==========================================
        if (lane == 0) {
            prefetch_tmap(&prm.tm_q); prefetch_tmap(&prm.tm_tq); prefetch_tmap(&prm.tm_k);
            prefetch_tmap(&prm.tm_tk); prefetch_tmap(&prm.tm_v); prefetch_tmap(&prm.tm_tv);
            uint32_t ring = 0, nq = 0;
            // this CTA's task list, assigned by the host head by head (assign_workers): all CTAs stream the same head's K, tK, V, tV
            // through L2 at the same time (a longest-first queue over ALL heads re-read them from DRAM 9.6 x: ncu, d = 64, 24 heads)
            int it = prm.pair_off[blockIdx.x];
            const int it_end = prm.pair_off[blockIdx.x + 1];
            for (uint32_t t = 0;; ++t) {
                const int ts = t & 1;
                wait(BAR_TASK_EMPTY + ts, ((t >> 1) & 1) ^ 1);
                const int task_id = (it < it_end && !sh->abort_flag) ? prm.pair_ids[it++] : prm.num_tasks;
                sh->task_id[ts] = task_id;
                mbar_arrive(bars + 8 * (BAR_TASK_FULL + ts));
                if (task_id >= prm.num_tasks) break;
                const aj_task task = prm.tasks[task_id];
                if (task.num_kv_tiles == 0) continue;
                // Q_i, tQ_i: two 64-column swizzle blocks each
                wait(BAR_Q_EMPTY, (nq & 1) ^ 1);
                mbar_expect_tx(bars + 8 * BAR_Q_FULL, PRIMAL ? Q_BYTES : 2 * Q_BYTES);
                tma_load_4d(sQ, &prm.tm_q, bars + 8 * BAR_Q_FULL, 0, task.q_begin, task.h, task.b);
                if (D == 128) tma_load_4d(sQ + QHALF_BYTES, &prm.tm_q, bars + 8 * BAR_Q_FULL, 64, task.q_begin, task.h, task.b);
                if (!PRIMAL) tma_load_4d(sTQ, &prm.tm_tq, bars + 8 * BAR_Q_FULL, 0, task.q_begin, task.h, task.b);
                if (!PRIMAL && D == 128) tma_load_4d(sTQ + QHALF_BYTES, &prm.tm_tq, bars + 8 * BAR_Q_FULL, 64, task.q_begin, task.h, task.b);
                ++nq;
                // ring order = MMA consumption order: KtK(0), KtK(1), VtV(0), KtK(2), VtV(1), ...
                // {K,tK} slot: [K h0 | tK h0 | K h1 | tK h1] so that [K ; tK] is one 128-row B operand per 64-column half;
                // {V,tV} slot: [V h0 | V h1 | tV h0 | tV h1] so that [V | tV] is one 256-column B operand.   (8 KB each)
                // D = 64: [K | tK] and [V | tV], one block per tensor.
                TileCursor ck, cv;
                ck.init(prm.k_begin, prm.k_end, task.range_begin, task.range_count);
                cv = ck;
                const int n = task.num_kv_tiles;
                auto push = [&](bool is_k) {
                    const uint32_t slot = ring % NSTAGE;
                    wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                    const uint32_t dst = sRing + slot * SLOT_BYTES, full = bars + 8 * (BAR_KV_FULL + slot);
                    mbar_expect_tx(full, PRIMAL ? SLOT_BYTES / 2 : SLOT_BYTES);
                    TileCursor &c = is_k ? ck : cv;
                    const CUtensorMap *m0 = is_k ? &prm.tm_k : &prm.tm_v, *m1 = is_k ? &prm.tm_tk : &prm.tm_tv;
                    const uint32_t o_m0h1 = is_k ? 2 * KVHALF_BYTES : KVHALF_BYTES;
                    const uint32_t o_m1h0 = D == 64 ? KVHALF_BYTES : is_k ? KVHALF_BYTES : 2 * KVHALF_BYTES;
                    const int row = c.key_row();
                    tma_load_4d(dst, m0, full, 0, row, task.h, task.b);
                    if (D == 128) tma_load_4d(dst + o_m0h1, m0, full, 64, row, task.h, task.b);
                    if (!PRIMAL) tma_load_4d(dst + o_m1h0, m1, full, 0, row, task.h, task.b);
                    if (!PRIMAL && D == 128) tma_load_4d(dst + 3 * KVHALF_BYTES, m1, full, 64, row, task.h, task.b);
                    c.next();
                    ++ring;
                };
                push(true);
                for (int j = 0; j < n; ++j) {
                    if (j + 1 < n) push(true);
                    push(false);
                }
            }
        }
    } else if (warp == 1) {
        // ================================================= MMA issuer ============================================
        // Every lane runs the control flow (so ring / tile counters and descriptors are warp-uniform and live in
        // uniform registers); the elected lane alone issues tcgen05.mma / tcgen05.commit.
        const bool leader = elect_one();
        const uint32_t q_lo = ((sQ >> 4) & 0x3FFF) | LBO_K, tq_lo = ((sTQ >> 4) & 0x3FFF) | LBO_K;
        uint32_t ring = 0, nq = 0, g = 0;   // g = tiles issued so far (selects S/tS buffer and barrier phase)
        auto issue_qk = [&](uint32_t gj) {
            const uint32_t slot = ring % NSTAGE;
            wait(BAR_KV_FULL + slot, (ring / NSTAGE) & 1);
            tc_fence_after();
            const uint32_t k_lo = (((sRing + slot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_K;
            const uint32_t tS_ = tmem + TM_S0 + (gj & 1) * TM_SBUF, tTS_ = tS_ + (TM_TS0 - TM_S0);
            if (leader) {
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t qoff = ((ks >> 2) * QHALF_BYTES + (ks & 3) * 32) >> 4;
                    const uint32_t koff = ((ks >> 2) * 2 * KVHALF_BYTES + (ks & 3) * 32) >> 4;
                    if (PRIMAL) {
                        mma_ss(tS_, q_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK1, ks > 0);   // S = Q K^T
                    } else {
                        mma_ss(tS_, q_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK2, ks > 0);   // [S | tS] = Q [K ; tK]^T
                        mma_ss(tTS_, tq_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK1, 1);      // tS += tQ K^T
                    }
                }
                tc_commit(bars + 8 * (BAR_KV_EMPTY + slot));
                tc_commit(bars + 8 * (BAR_S_FULL + (gj & 1)));
            }
            __syncwarp();
            ++ring;
        };
        for (uint32_t t = 0;; ++t) {
            const int ts = t & 1;
            wait(BAR_TASK_FULL + ts, (t >> 1) & 1);
            const int task_id = (int)warp_uniform((uint32_t)sh->task_id[ts] | (sh->abort_flag ? 0x40000000u : 0u));
            if (leader) mbar_arrive(bars + 8 * (BAR_TASK_EMPTY + ts));
            if (task_id >= prm.num_tasks) break;
            const int n = (int)warp_uniform((uint32_t)prm.tasks[task_id].num_kv_tiles);
            if (n == 0) continue;
            wait(BAR_Q_FULL, nq & 1);
            ++nq;
            tc_fence_after();
            issue_qk(g);
            for (int j = 0; j < n; ++j) {
                const uint32_t gj = g + j, b = gj & 1;
                if (j + 1 < n) issue_qk(gj + 1);
                else if (leader) tc_commit(bars + 8 * BAR_Q_EMPTY);   // every QK of this task has been issued
                const uint32_t slot = ring % NSTAGE;
                // V tile in smem: key row r at r*128 bytes inside each 64-column block; 16-key K steps are 2 KB apart.
                const uint32_t v_lo = (((sRing + slot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_V;
                const uint32_t tP = tmem + TM_S0 + b * TM_SBUF, tH = tP + (TM_TS0 - TM_S0);
                const uint32_t acc = j > 0 ? 1u : 0u;
                wait(BAR_P_FULL + b, (gj >> 1) & 1);
                wait(BAR_KV_FULL + slot, (ring / NSTAGE) & 1);
                tc_fence_after();
                if (leader) {
#pragma unroll
                    for (int ks = 0; ks < BC / 16; ++ks)    // [O | T] += P~ [V | tV]; PRIMAL: O += P~ V
                        mma_ts(tmem + TM_O, tP + ks * 8, v_lo + ks * (2048 >> 4), DESC_HI, PRIMAL ? IDESC_PV1 : IDESC_PV2, acc | (ks > 0));
                }
                __syncwarp();
                if (!PRIMAL) {
                    wait(BAR_H_FULL + b, (gj >> 1) & 1);
                    tc_fence_after();
                }
                if (leader) {
#pragma unroll
                    for (int ks = 0; ks < BC / 16; ++ks)    // T += H~ V
                        if (!PRIMAL) mma_ts(tmem + TM_T, tH + ks * 8, v_lo + ks * (2048 >> 4), DESC_HI, IDESC_PV1, 1);
                    tc_commit(bars + 8 * (BAR_KV_EMPTY + slot));
                    tc_commit(bars + 8 * (BAR_PV_DONE + b));
                }
                __syncwarp();
                ++ring;
            }
            g += n;
        }
    } else if (warp >= 4) {
        // ================================================= softmax / tangent weights / epilogue ==================
        const int row = threadIdx.x - 128;                       // query row inside the tile = TMEM lane
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const float sl2 = prm.scale_log2, sc = prm.scale;
        const uint64_t sl2_2 = pack2(sl2, sl2), sc_2 = pack2(sc, sc);
        uint32_t g = 0;
        for (uint32_t t = 0;; ++t) {
            const int ts = t & 1;
            wait(BAR_TASK_FULL + ts, (t >> 1) & 1);
            const int task_id = sh->task_id[ts];
            __syncwarp();
            if (lane == 0) mbar_arrive(bars + 8 * (BAR_TASK_EMPTY + ts));
            if (task_id >= prm.num_tasks || sh->abort_flag) break;
            const aj_task task = prm.tasks[task_id];
            const int n = task.num_kv_tiles;
            float m_ref = M_UNSET;
            uint64_t l2[2] = {0ull, 0ull}, r2[2] = {0ull, 0ull};   // 4 partial sums each of l = sum P~ and r = sum H~
            TileCursor cur;
            cur.init(prm.k_begin, prm.k_end, task.range_begin, task.range_count);
            int cur_entry = -1, row_lo = 0, row_hi = 0;
            for (int j = 0; j < n; ++j, cur.next()) {
                const uint32_t gj = g + j, b = gj & 1;
                const uint32_t tS_ = tmem + lane_base + TM_S0 + b * TM_SBUF, tTS_ = tS_ + (TM_TS0 - TM_S0);
                if (cur.entry() != cur_entry) {                    // rows of this tile that may see the entry's keys
                    cur_entry = cur.entry();
                    const uint32_t rr = prm.rows[cur_entry];
                    row_lo = (int)(rr & 0xffffu); row_hi = (int)((rr >> 16) & 0x7fffu);   // bit 31: key-tangents-zero flag (CTA-pair kernel)
                }
                wait(BAR_S_FULL + b, (gj >> 1) & 1);
                tc_fence_after();
                uint32_t su[2][32], tu[2][32];
                tmem_ld32(tS_, su[0]);
                tmem_ld32(tS_ + 32, su[1]);
                tc_wait_ld(su[0], su[1]);
                if (!PRIMAL) {
                    tmem_ld32(tTS_, tu[0]);                        // in flight while P~ is computed
                    tmem_ld32(tTS_ + 32, tu[1]);
                }
                // tile-valid mask: S = -inf past the entry's last key and on rows outside its row interval
                const int valid = (row >= row_lo && row < row_hi) ? cur.valid() : 0;
                if (valid < BC) {
#pragma unroll
                    for (int c = 0; c < BC; ++c) if (c >= valid) su[c >> 5][c & 31] = 0xff800000u;
                }
                float mx[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) mx[i] = __uint_as_float(su[0][i]);
#pragma unroll
                for (int c = 4; c < BC; ++c) mx[c & 3] = fmaxf(mx[c & 3], __uint_as_float(su[c >> 5][c & 31]));
                const float cand = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * sl2;
                {
                    // Lazy reference max (PAPER.md:922-927 applied only when needed).  A row whose reference is still
                    // unset has O = T = l = r = 0 exactly, so it adopts the tile max with nothing to rescale.
                    const bool need = cand > m_ref + RESCALE_THRESHOLD;
                    const bool fresh = m_ref == M_UNSET;
                    if (__any_sync(0xffffffffu, need && !fresh)) {
                        // e^{m - m_new} applied to O, T (= A + B), l, r; needs PV(j-1) finished
                        const uint32_t gp = gj - 1;
                        wait(BAR_PV_DONE + (gp & 1), (gp >> 1) & 1);
                        tc_fence_after();
                        const float f = (need && !fresh) ? ex2(m_ref - cand) : 1.f;
#pragma unroll 1
                        for (int cb = 0; cb < (PRIMAL ? D : 2 * D); cb += 32) {
                            uint32_t a[32];
                            tmem_ld32(tmem + lane_base + cb, a);
                            tc_wait_ld(a);
#pragma unroll
                            for (int c = 0; c < 32; ++c) a[c] = __float_as_uint(__uint_as_float(a[c]) * f);
                            tmem_st32(tmem + lane_base + cb, a);
                        }
                        const uint64_t f2 = pack2(f, f);
                        l2[0] = fmul2(l2[0], f2); l2[1] = fmul2(l2[1], f2);
                        r2[0] = fmul2(r2[0], f2); r2[1] = fmul2(r2[1], f2);
                    }
                    if (need) m_ref = cand;
                }
                // P~ = exp2(S*s*log2e - m_ref); l += rowsum
                const uint64_t negm2 = pack2(-m_ref, -m_ref);
                float p[BC];
                {
                    uint32_t pk[32];
#pragma unroll
                    for (int c = 0; c < BC / 2; ++c) {
                        const uint64_t x = ffma2(pack2(su[c >> 4][(2 * c) & 31], su[c >> 4][(2 * c + 1) & 31]), sl2_2, negm2);
                        float x0, x1;
                        unpack2(x, x0, x1);
                        p[2 * c] = ex2(x0); p[2 * c + 1] = ex2(x1);
                        l2[c & 1] = fadd2(l2[c & 1], pack2(p[2 * c], p[2 * c + 1]));
                        pk[c] = pack_bf16(p[2 * c], p[2 * c + 1]);
                    }
                    tmem_st32(tS_, pk);
                }
                tc_wait_st();
                tc_fence_before();
                mbar_arrive(bars + 8 * (BAR_P_FULL + b));
                // H~ = P~ o (s * tS); r += rowsum.  Masked columns have P~ = 0, so H~ = 0.
                if (PRIMAL) continue;
                tc_wait_ld(tu[0], tu[1]);
                {
                    uint32_t hk[32];
#pragma unroll
                    for (int c = 0; c < BC / 2; ++c) {
                        const uint64_t tsc = fmul2(pack2(tu[c >> 4][(2 * c) & 31], tu[c >> 4][(2 * c + 1) & 31]), sc_2);
                        const uint64_t h = fmul2(pack2(p[2 * c], p[2 * c + 1]), tsc);
                        r2[c & 1] = fadd2(r2[c & 1], h);
                        float h0, h1;
                        unpack2(h, h0, h1);
                        hk[c] = pack_bf16(h0, h1);
                    }
                    tmem_st32(tTS_, hk);
                }
                tc_wait_st();
                tc_fence_before();
                mbar_arrive(bars + 8 * (BAR_H_FULL + b));
            }
            // ---- epilogue (Eq. 45) ----
            const bool store = row < task.q_rows;
            const int64_t grow = task.q_begin + row;
            __nv_bfloat16 *op = (__nv_bfloat16 *)prm.o.ptr + task.b * prm.o.stride_b + task.h * prm.o.stride_h + grow * prm.o.stride_n;
            __nv_bfloat16 *tp = (__nv_bfloat16 *)prm.to.ptr + task.b * prm.to.stride_b + task.h * prm.to.stride_h + grow * prm.to.stride_n;
            if (n == 0) {                                         // no key: O = 0, tO = 0, lse = -inf (R9)
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = 0; c < D / 8; ++c) { ((uint4 *)op)[c] = z; if (prm.to.ptr) ((uint4 *)tp)[c] = z; }
                    if (prm.lse) prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = -INFINITY;
                    if (prm.tlse) prm.tlse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = 0.f;
                }
                continue;
            }
            {
                const uint32_t gl = g + n - 1;
                wait(BAR_PV_DONE + (gl & 1), (gl >> 1) & 1);
                tc_fence_after();
            }
            float la, lb, lc, ld, ra, rb, rc, rd;
            unpack2(l2[0], la, lb); unpack2(l2[1], lc, ld);
            unpack2(r2[0], ra, rb); unpack2(r2[1], rc, rd);
            const float l = (la + lb) + (lc + ld), r = (ra + rb) + (rc + rd);
            const float inv = l > 0.f ? 1.f / l : 0.f, rl = r * inv;   // l = 0: the row saw no key (O = 0, tO = 0, lse = -inf)
#pragma unroll 1
            for (int cb = 0; cb < D; cb += 32) {
                uint32_t ao[32], at[32];
                tmem_ld32(tmem + lane_base + TM_O + cb, ao);
                if (PRIMAL) {
                    tc_wait_ld(ao);
#pragma unroll
                    for (int c = 0; c < 32; ++c) at[c] = 0u;
                } else {
                    tmem_ld32(tmem + lane_base + TM_T + cb, at);
                    tc_wait_ld(ao, at);
                }
                if (store) {
#pragma unroll
                    for (int v4 = 0; v4 < 4; ++v4) {
                        uint32_t wo[4], wt[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int c = v4 * 8 + 2 * e;
                            const float o0 = __uint_as_float(ao[c]) * inv, o1 = __uint_as_float(ao[c + 1]) * inv;
                            const float t0 = fmaf(__uint_as_float(at[c]), inv, -rl * o0);
                            const float t1 = fmaf(__uint_as_float(at[c + 1]), inv, -rl * o1);
                            wo[e] = pack_bf16(o0, o1);
                            wt[e] = pack_bf16(t0, t1);
                        }
                        *(uint4 *)(op + cb + v4 * 8) = make_uint4(wo[0], wo[1], wo[2], wo[3]);
                        if (!PRIMAL || prm.to.ptr) *(uint4 *)(tp + cb + v4 * 8) = make_uint4(wt[0], wt[1], wt[2], wt[3]);
                    }
                }
            }
            if (store && prm.lse)
                prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = l > 0.f ? (m_ref + log2f(l)) * 0.6931471805599453f : -INFINITY;
            if (store && prm.tlse) prm.tlse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = rl;   // r / l
            tc_fence_before();
            g += n;
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    }
}

}  // namespace

size_t umma_smem_bytes() { return Cfg<128>::SMEM_TOTAL; }

cudaError_t launch_umma(const UmmaParams &prm, int d, bool primal, int grid, cudaStream_t stream) {
    if (grid <= 0) return cudaSuccess;
    static std::atomic<uint64_t> configured[4];
    auto run = [&](auto kernel, uint32_t smem, std::atomic<uint64_t> &done) -> cudaError_t {
        if (cudaError_t e = ensure_dynamic_smem(kernel, (int)smem, done)) return e;
        kernel<<<grid, NTHREADS, smem, stream>>>(prm);
        return cudaGetLastError();
    };
    if (d == 64) return primal ? run(attn_jvp_umma_kernel<64, true>, Cfg<64>::SMEM_TOTAL, configured[1])
                               : run(attn_jvp_umma_kernel<64, false>, Cfg<64>::SMEM_TOTAL, configured[0]);
    if (d == 128) return primal ? run(attn_jvp_umma_kernel<128, true>, Cfg<128>::SMEM_TOTAL, configured[3])
                                : run(attn_jvp_umma_kernel<128, false>, Cfg<128>::SMEM_TOTAL, configured[2]);
    return cudaErrorInvalidValue;
}

}  // namespace aj
