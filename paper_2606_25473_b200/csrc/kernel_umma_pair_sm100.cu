// bf16 attention + JVP for sm_100a on CTA PAIRS: TMA -> shared-memory ring -> tcgen05.mma.cta_group::2 (M = 256).
//
// Same computation as kernel_umma_sm100.cu (Algorithm 1), re-tiled so that every shared-memory
// operand MMA has N = 128 and the two SMs of a pair share the K/V stream:
//   task      = 256 query rows of one (b, h): CTA 0 of the pair owns rows [0,128), CTA 1 rows [128,256)
//   pair-step = TWO 64-key tiles j0 = 2p, j1 = 2p+1 of the task's key stream
//     [S(j0) | S(j1)]    = Q  [K(j0) ; K(j1)]^T                       8 x (M256 N128 K16), A and B from shared memory
//     [tS(j0) | tS(j1)]  = Q  [tK(j0) ; tK(j1)]^T + tQ [K(j0) ; K(j1)]^T   16 x                      (Eq. 42-43)
//     per tile: O += P~ V, T += P~ tV, T += H~ V                      3 x 4 x (M256 N128 K16), A = bf16 P~/H~ in TMEM
//   The B operand of a cta_group::2 MMA is split by N between the two CTAs: CTA c stages K(j_c) and tK(j_c) (all 128
//   columns) and the column half [64c, 64c+64) of V and tV of both tiles.  Per 64-key tile and SM this is 32 KB of TMA
//   writes and 96 KB of operand reads (single-CTA kernel: 64 KB and 160 KB), which leaves the 128 B/clk shared-memory
//   port under the 1536 clk of tensor math; and no instruction has the A-operand-bound N = 64 shape.
//   S/tS are single-buffered (TMEM: O 128 | T 128 | S 2x64 | tS 2x64 columns); the overlap comes from the order inside
//   a pair-step: softmax turns S into P~ while the tensor pipe computes tS, and tS into H~ while it runs the P~ MMAs.
//   The lazy reference max (kernel_umma_sm100.cu) is moved once per pair-step, from the max over both tiles.
// Roles per CTA (8 warps): warp 0 TMA producer, warp 1 MMA issuer (CTA 0 only), warp 2 TMEM allocator, warps 4-7
// softmax / tangent weights / rescale / epilogue (thread = query row = TMEM lane).  Tasks are assigned to pairs by the
// host (longest-processing-time first), so there is no device-side work queue.
//
// Structural-zero tangents (aj_tangent_zero; "The tangent of the clean context is zero"):
//   key-zero pair-step (both tiles' tK, tV are zero, schedule entry flag): tK, tV are not loaded, Q tK^T and P~ tV are not
//     issued: 32 MMAs instead of 48.  The producer decides per pair-step and tells the MMA warp through `slot_kz`.
//   primal-only task (AJ_TASK_PRIMAL_ONLY: tQ of its rows is zero too): only S = Q K^T and O += P~ V (16 MMAs per
//     pair-step); the tS columns of TMEM become a second S buffer, so that S(p+2) is computed while the softmax of
//     pair-step p+1 runs (the classic two-stage forward-attention pipeline); tO of its rows is written as 0.
// Barrier phases are counted per barrier set: c_s (S_FULL, P_FULL), c_ts (TS_FULL, H_FULL), c_pv (PV_DONE); every role
// walks the same task list, so the counts agree.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

#include "kernels.hpp"
#include "pair_common.cuh"
#include "umma_ptx.cuh"

namespace aj {

namespace {

using namespace ptx;
using pairk::PairWaiter;
using pairk::RowCursor;
using pairk::Tile;
using pairk::TileCursor;

constexpr int BR = 128;                // query rows per CTA (UMMA M = 256 over the pair)
using pairk::BC;                       // 64 keys per tile
constexpr int D = 128;
constexpr int NSTAGE = 5;              // ring slots of 32 KB
constexpr uint32_t Q_BYTES = BR * D * 2;           // 32 KB
constexpr uint32_t QHALF_BYTES = BR * 64 * 2;      // 16 KB: one 64-column swizzle block of Q
constexpr uint32_t BLK_BYTES = BC * 64 * 2;        // 8 KB: 64 keys x 64 columns, 128-byte swizzled rows
constexpr uint32_t SLOT_BYTES = 4 * BLK_BYTES;     // 32 KB
constexpr uint32_t SMEM_TILES = 2 * Q_BYTES + NSTAGE * SLOT_BYTES;  // 224 KB
constexpr uint32_t SMEM_TOTAL = SMEM_TILES + 1024 /*align*/ + 256 /*barriers*/;
constexpr int NTHREADS = 256;

constexpr uint32_t TM_O = 0, TM_T = 128, TM_S = 256, TM_TS = 384;   // S(j_i) at TM_S + 64 i, tS(j_i) at TM_TS + 64 i
constexpr float RESCALE_THRESHOLD = 8.0f;  // log2 units
constexpr float M_UNSET = -1.0e30f;

enum {
    BAR_Q_FULL = 0,                         // CTA 0: Q, tQ of both CTAs landed (transaction bytes of both)
    BAR_Q_EMPTY,                            // both: every QK MMA of the task is complete
    BAR_KV_FULL,                            // CTA 0: ring slot filled in both CTAs
    BAR_KV_EMPTY = BAR_KV_FULL + NSTAGE,    // both: the MMAs reading the slot are complete
    BAR_S_FULL = BAR_KV_EMPTY + NSTAGE,     // both: [S(j0) | S(j1)] complete
    BAR_TS_FULL,                            // both: [tS(j0) | tS(j1)] complete
    BAR_P_FULL,                             // CTA 0, x2: P~(j_i) stored by all 8 softmax warps of the pair
    BAR_H_FULL = BAR_P_FULL + 2,            // CTA 0, x2: H~(j_i)
    BAR_PV_DONE = BAR_H_FULL + 2,           // both: every MMA into O, T of the pair-step is complete
    NUM_BARS
};

// Instruction descriptor, kind::f16: D fp32, A and B bf16, N >> 3 at bit 17, M >> 4 at bit 24 (M = 256 over the pair).
constexpr uint32_t make_idesc(int n, bool b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}
constexpr uint32_t IDESC_QK = make_idesc(2 * BC, false);   // 256 x 128 x 16, B K-major (64 key rows per CTA)
constexpr uint32_t IDESC_PV = make_idesc(D, true);         // 256 x 128 x 16, B MN-major (64 columns per CTA)
constexpr uint32_t DESC_HI = desc_hi(1024);                // 8-row / 8-key groups are 1024 B apart
constexpr uint32_t LBO_CANON = desc_lo_lbo(16);            // single 64-column block per operand: LBO unused

struct Shared {
    uint64_t bars[NUM_BARS];
    uint32_t tmem_base;
    int abort_flag;
    int slot_kz[NSTAGE];   // leader CTA: the pair-step whose {K, tK} sits in the slot has zero key tangents (set by the
                           // producer before it arms KV_FULL[slot], read by the MMA warp after its wait)
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
attn_jvp_umma_pair_kernel(const __grid_constant__ UmmaParams prm) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;       // 1024-byte alignment for the 128-byte swizzle
    Shared *sh = reinterpret_cast<Shared *>(smem_raw + (tiles - raw) + SMEM_TILES);
    const uint32_t sQ = tiles, sTQ = tiles + Q_BYTES, sRing = tiles + 2 * Q_BYTES;
    const uint32_t bars = smem_u32(sh->bars);
    const PairWaiter wait{bars, &sh->abort_flag, prm.counters + 2, 100};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();              // 0 = leader (issues the MMAs, owns the "full" barriers)
    const uint32_t lead_bars = mapa(bars, 0);             // the leader's barrier array in the cluster window
    const int pair = blockIdx.x >> 1;
    const int list_begin = prm.pair_off[pair], list_end = prm.pair_off[pair + 1];

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * BAR_Q_FULL, 1);
        mbar_init(bars + 8 * BAR_Q_EMPTY, 1);
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bars + 8 * (BAR_KV_FULL + i), 1); mbar_init(bars + 8 * (BAR_KV_EMPTY + i), 1); }
        mbar_init(bars + 8 * BAR_S_FULL, 1);
        mbar_init(bars + 8 * BAR_TS_FULL, 1);
        for (int i = 0; i < 2; ++i) {
            mbar_init(bars + 8 * (BAR_P_FULL + i), 8);    // one arrive per softmax warp of the pair
            mbar_init(bars + 8 * (BAR_H_FULL + i), 8);
        }
        mbar_init(bars + 8 * BAR_PV_DONE, 1);
        sh->abort_flag = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sh->tmem_base)), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    cluster_arrive();                                     // the peer's barriers are initialised before anyone signals them
    cluster_wait();
    tc_fence_after();
    const uint32_t tmem = sh->tmem_base;

    if (warp == 0) {
        // ================================================= TMA producer (both CTAs) ================================
        if (lane == 0) {
            prefetch_tmap(&prm.tm_q); prefetch_tmap(&prm.tm_tq); prefetch_tmap(&prm.tm_k);
            prefetch_tmap(&prm.tm_tk); prefetch_tmap(&prm.tm_v); prefetch_tmap(&prm.tm_tv);
            uint32_t ring = 0, nq = 0;
            int sync_prev = -1;
            bool sync_on = true;
            int sync_fail = 0;
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task task = prm.tasks[prm.pair_ids[it]];
                const int n = task.num_kv_tiles;
                if (n == 0 || sh->abort_flag) continue;
                if (prm.slot_sync && sync_on) {
                    // Task-slot rendezvous of the producers (uniform-cost schedules only): the pairs start every slot together, so they
                    // stream the same keys of the same head at the same time and L2 serves all but one of them.  Without it the pairs
                    // drift apart by a fraction of a per cent per task, and after a few dozen slots every pair streams from DRAM on its
                    // own (full mask, N = 115,200, 24 heads: 379 GB of DRAM reads per launch for 5.7 GB of inputs).  Bounded: after
                    // ~0.1 ms the pair goes on alone (the rendezvous is a performance hint, never a correctness condition).
                    // Per-head mode (tasks of different cost): the pairs meet when they enter a head -- the lists are built for that
                    // (assign_workers levels the workers at every head), so the wait is the imbalance inside one head, about one
                    // short task; the bound is correspondingly longer.
                    const int slot_i = prm.sync_per_head ? task.b * prm.H + task.h : it - list_begin;
                    if (!prm.sync_per_head || slot_i != sync_prev) {
                        if (rank == 0) atomicAdd(prm.slot_sync + slot_i, 1);
                        const int want = prm.slot_expect[slot_i];
                        const long long t0 = clock64();
                        const long long limit = prm.sync_per_head ? 1500000 : 400000;
                        while (*(volatile int32_t *)(prm.slot_sync + slot_i) < want && clock64() - t0 < limit) __nanosleep(64);
                        // Rendezvous that keep timing out mean that the pairs are not all running (other kernels hold SMs, or two launches
                        // share the counters): after three in a row this pair stops waiting for the rest of the launch.
                        if (*(volatile int32_t *)(prm.slot_sync + slot_i) < want) { if (++sync_fail >= 3) sync_on = false; } else sync_fail = 0;
                        sync_prev = slot_i;
                    }
                }
                const bool primal = (task.flags & AJ_TASK_PRIMAL_ONLY) != 0;
                // Q_i, tQ_i: this CTA's 128 rows, two 64-column swizzle blocks each (no tQ if it is zero)
                wait(BAR_Q_EMPTY, (nq & 1) ^ 1);
                const uint32_t qfull = lead_bars + 8 * BAR_Q_FULL;
                if (rank == 0) mbar_expect_tx(bars + 8 * BAR_Q_FULL, primal ? 2 * Q_BYTES : 4 * Q_BYTES);
                const int qrow = task.q_begin + BR * (int)rank;
                tma_load_4d_pair(sQ, &prm.tm_q, qfull, 0, qrow, task.h, task.b);
                tma_load_4d_pair(sQ + QHALF_BYTES, &prm.tm_q, qfull, 64, qrow, task.h, task.b);
                if (!primal) {
                    tma_load_4d_pair(sTQ, &prm.tm_tq, qfull, 0, qrow, task.h, task.b);
                    tma_load_4d_pair(sTQ + QHALF_BYTES, &prm.tm_tq, qfull, 64, qrow, task.h, task.b);
                }
                ++nq;
                TileCursor cur;
                cur.init(prm.k_begin, prm.k_end, task.range_begin, task.range_count);
                const int np = (n + 1) >> 1;
                int flag_entry = -1;
                bool flag = false;                         // tK, tV of the entry's keys are structurally zero
                auto entry_kz = [&](int e) { if (e != flag_entry) { flag_entry = e; flag = (prm.rows[e] >> 31) != 0; } return flag; };
                for (int p = 0; p < np; ++p) {
                    const Tile t0 = cur.get();
                    cur.next();
                    Tile t1 = t0;                          // odd tail: the second tile is a fully masked copy of the first
                    bool kz = primal || entry_kz(t0.entry);
                    if (2 * p + 1 < n) { t1 = cur.get(); cur.next(); kz = kz && (primal || entry_kz(t1.entry)); }
                    const uint32_t slot_tx = kz ? SLOT_BYTES : 2 * SLOT_BYTES;   // bytes of both CTAs
                    {   // {K, tK} of this CTA's tile: [K h0 | K h1 | tK h0 | tK h1]
                        const uint32_t slot = ring % NSTAGE;
                        wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                        const uint32_t dst = sRing + slot * SLOT_BYTES, full = lead_bars + 8 * (BAR_KV_FULL + slot);
                        if (rank == 0) {
                            ((volatile int *)sh->slot_kz)[slot] = kz ? 1 : 0;
                            mbar_expect_tx(bars + 8 * (BAR_KV_FULL + slot), slot_tx);
                        }
                        const int row = rank ? t1.key_row : t0.key_row;
                        tma_load_4d_pair(dst, &prm.tm_k, full, 0, row, task.h, task.b);
                        tma_load_4d_pair(dst + BLK_BYTES, &prm.tm_k, full, 64, row, task.h, task.b);
                        if (!kz) {
                            tma_load_4d_pair(dst + 2 * BLK_BYTES, &prm.tm_tk, full, 0, row, task.h, task.b);
                            tma_load_4d_pair(dst + 3 * BLK_BYTES, &prm.tm_tk, full, 64, row, task.h, task.b);
                        }
                        ++ring;
                    }
                    {   // this CTA's column half of {V, tV} of both tiles: [V(j0) | tV(j0) | V(j1) | tV(j1)]
                        const uint32_t slot = ring % NSTAGE;
                        wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                        const uint32_t dst = sRing + slot * SLOT_BYTES, full = lead_bars + 8 * (BAR_KV_FULL + slot);
                        if (rank == 0) mbar_expect_tx(bars + 8 * (BAR_KV_FULL + slot), slot_tx);
                        const int col = 64 * (int)rank;
                        tma_load_4d_pair(dst, &prm.tm_v, full, col, t0.key_row, task.h, task.b);
                        tma_load_4d_pair(dst + 2 * BLK_BYTES, &prm.tm_v, full, col, t1.key_row, task.h, task.b);
                        if (!kz) {
                            tma_load_4d_pair(dst + BLK_BYTES, &prm.tm_tv, full, col, t0.key_row, task.h, task.b);
                            tma_load_4d_pair(dst + 3 * BLK_BYTES, &prm.tm_tv, full, col, t1.key_row, task.h, task.b);
                        }
                        ++ring;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================================================= MMA issuer (leader CTA) ==================================
        // Every lane runs the control flow (counters and descriptors stay warp-uniform), one elected lane issues.
        if (rank == 0) {
            const bool leader = elect_one();
            const uint32_t q_lo = ((sQ >> 4) & 0x3FFF) | LBO_CANON, tq_lo = ((sTQ >> 4) & 0x3FFF) | LBO_CANON;
            uint32_t ring = 0, nq = 0, c_s = 0, c_ts = 0;   // ring items consumed; uses of the S / tS barrier sets
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task &tk = prm.tasks[prm.pair_ids[it]];
                const int n = (int)warp_uniform((uint32_t)tk.num_kv_tiles | (sh->abort_flag ? 0x80000000u : 0u));
                if (n <= 0) continue;
                const bool primal = warp_uniform((uint32_t)tk.flags & AJ_TASK_PRIMAL_ONLY) != 0;
                wait(BAR_Q_FULL, nq & 1);
                ++nq;
                tc_fence_after();
                const int np = (n + 1) >> 1;
                if (primal) {
                    // ---- primal-only task: S double-buffered in the S and tS columns; ring items: K(p) = base + 2p, V(p) = base + 2p + 1
                    const uint32_t base = ring;
                    ring += 2 * (uint32_t)np;
                    auto issue_S = [&](int p) {
                        const uint32_t item = base + 2 * (uint32_t)p, slot = item % NSTAGE;
                        wait(BAR_KV_FULL + slot, (item / NSTAGE) & 1);
                        tc_fence_after();
                        const uint32_t k_lo = (((sRing + slot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
                        const uint32_t tS = tmem + ((p & 1) ? TM_TS : TM_S);
                        if (leader) {
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks) {   // [S(j0) | S(j1)] = Q [K(j0) ; K(j1)]^T
                                const uint32_t qoff = ((ks >> 2) * QHALF_BYTES + (ks & 3) * 32) >> 4;
                                const uint32_t koff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                                mma_ss_pair(tS, q_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK, ks > 0);
                            }
                            tc_commit_pair(bars + 8 * ((p & 1) ? BAR_TS_FULL : BAR_S_FULL), 3);
                            tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + slot), 3);
                            if (p + 1 == np) tc_commit_pair(bars + 8 * BAR_Q_EMPTY, 3);
                        }
                        __syncwarp();
                    };
                    issue_S(0);
                    if (np > 1) issue_S(1);
                    for (int p = 0; p < np; ++p) {
                        const uint32_t item = base + 2 * (uint32_t)p + 1, vslot = item % NSTAGE;
                        wait(BAR_KV_FULL + vslot, (item / NSTAGE) & 1);
                        const uint32_t v_lo = (((sRing + vslot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
                        const int buf = p & 1;
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const uint32_t vi_lo = v_lo + ((2 * i * BLK_BYTES) >> 4);
                            const uint32_t tP = tmem + (buf ? TM_TS : TM_S) + i * BC;
                            const uint32_t acc = (p > 0 || i > 0) ? 1u : 0u;
                            wait((buf ? BAR_H_FULL : BAR_P_FULL) + i, (buf ? c_ts : c_s) & 1);
                            tc_fence_after();
                            if (leader) {
#pragma unroll
                                for (int ks = 0; ks < BC / 16; ++ks)    // O += P~ V
                                    mma_ts_pair(tmem + TM_O, tP + ks * 8, vi_lo + ks * (2048 >> 4), DESC_HI, IDESC_PV, acc | (ks > 0));
                            }
                            __syncwarp();
                        }
                        if (leader) {
                            tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + vslot), 3);
                            tc_commit_pair(bars + 8 * BAR_PV_DONE, 3);
                        }
                        __syncwarp();
                        if (buf) ++c_ts; else ++c_s;
                        if (p + 2 < np) issue_S(p + 2);       // overwrites P~(p): the pipe executes in order
                    }
                    continue;
                }
                // ---- general task.  QK of pair-step p: [S | S] first (softmax starts on it), then [tS | tS]
                uint32_t kslot = 0, k_lo = 0;
                bool kz_next = false;                    // key tangents of the pair-step whose S was issued last are zero
                uint32_t t_acc = 0;                      // T has been written in this task
                auto issue_s = [&]() {
                    kslot = ring % NSTAGE;
                    wait(BAR_KV_FULL + kslot, (ring / NSTAGE) & 1);
                    tc_fence_after();
                    k_lo = (((sRing + kslot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
                    if (leader) {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {   // [S(j0) | S(j1)] = Q [K(j0) ; K(j1)]^T
                            const uint32_t qoff = ((ks >> 2) * QHALF_BYTES + (ks & 3) * 32) >> 4;
                            const uint32_t koff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                            mma_ss_pair(tmem + TM_S, q_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK, ks > 0);
                        }
                        tc_commit_pair(bars + 8 * BAR_S_FULL, 3);
                    }
                    __syncwarp();
                    // read after the S MMAs are on their way: only tS and the P~ tV MMAs of this pair-step depend on it
                    kz_next = warp_uniform((uint32_t)((volatile int *)sh->slot_kz)[kslot]) != 0;
                    ++ring;
                };
                auto issue_ts = [&](bool last) {
                    const uint32_t tk_lo = k_lo + ((2 * BLK_BYTES) >> 4);
                    if (leader) {
                        if (!kz_next) {
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks) {   // [tS(j0) | tS(j1)] = Q [tK ; tK]^T + tQ [K ; K]^T  (Eq. 43)
                                const uint32_t qoff = ((ks >> 2) * QHALF_BYTES + (ks & 3) * 32) >> 4;
                                const uint32_t koff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                                mma_ss_pair(tmem + TM_TS, q_lo + qoff, DESC_HI, tk_lo + koff, DESC_HI, IDESC_QK, ks > 0);
                            }
                        }
                        const uint32_t acc0 = kz_next ? 0u : 1u;    // tK = 0: tS = tQ K^T alone
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            const uint32_t qoff = ((ks >> 2) * QHALF_BYTES + (ks & 3) * 32) >> 4;
                            const uint32_t koff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                            mma_ss_pair(tmem + TM_TS, tq_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK, acc0 | (ks > 0));
                        }
                        tc_commit_pair(bars + 8 * BAR_TS_FULL, 3);
                        tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + kslot), 3);
                        if (last) tc_commit_pair(bars + 8 * BAR_Q_EMPTY, 3);   // every QK of this task has been issued
                    }
                    __syncwarp();
                };
                issue_s();
                issue_ts(np == 1);
                for (int p = 0; p < np; ++p, ++c_s, ++c_ts) {
                    // Issue order P~(j0), P~(j1), S of the NEXT pair-step, H~(j0), H~(j1), tS of the next pair-step: the
                    // tensor pipe executes in order, so S(p+1) may overwrite P~(p) and tS(p+1) may overwrite H~(p), and
                    // the softmax of step p+1 runs while the pipe does the H~ MMAs and tS(p+1).
                    const bool kz = kz_next;                // this pair-step: tV = 0, so T += P~ tV is skipped
                    const uint32_t vslot = ring % NSTAGE;
                    wait(BAR_KV_FULL + vslot, (ring / NSTAGE) & 1);
                    ++ring;
                    // [V(j0) | tV(j0) | V(j1) | tV(j1)], this CTA's 64 columns: key r at r*128 B, 16-key K steps 2 KB apart
                    const uint32_t v_lo = (((sRing + vslot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const uint32_t vi_lo = v_lo + ((2 * i * BLK_BYTES) >> 4), tvi_lo = vi_lo + (BLK_BYTES >> 4);
                        const uint32_t tP = tmem + TM_S + i * BC;
                        const uint32_t acc = (p > 0 || i > 0) ? 1u : 0u;
                        wait(BAR_P_FULL + i, c_s & 1);
                        tc_fence_after();
                        if (leader) {
#pragma unroll
                            for (int ks = 0; ks < BC / 16; ++ks)    // O += P~ V
                                mma_ts_pair(tmem + TM_O, tP + ks * 8, vi_lo + ks * (2048 >> 4), DESC_HI, IDESC_PV, acc | (ks > 0));
                            if (!kz) {
#pragma unroll
                                for (int ks = 0; ks < BC / 16; ++ks)    // T += P~ tV
                                    mma_ts_pair(tmem + TM_T, tP + ks * 8, tvi_lo + ks * (2048 >> 4), DESC_HI, IDESC_PV, t_acc | (ks > 0));
                            }
                        }
                        if (!kz) t_acc = 1;
                        __syncwarp();
                    }
                    if (p + 1 < np) issue_s();
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const uint32_t vi_lo = v_lo + ((2 * i * BLK_BYTES) >> 4);
                        const uint32_t tH = tmem + TM_TS + i * BC;
                        wait(BAR_H_FULL + i, c_ts & 1);
                        tc_fence_after();
                        if (leader) {
#pragma unroll
                            for (int ks = 0; ks < BC / 16; ++ks)    // T += H~ V
                                mma_ts_pair(tmem + TM_T, tH + ks * 8, vi_lo + ks * (2048 >> 4), DESC_HI, IDESC_PV, t_acc | (ks > 0));
                        }
                        t_acc = 1;
                        __syncwarp();
                    }
                    if (leader) {
                        tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + vslot), 3);
                        tc_commit_pair(bars + 8 * BAR_PV_DONE, 3);
                    }
                    __syncwarp();
                    if (p + 1 < np) issue_ts(p + 2 == np);
                }
            }
        }
    } else if (warp >= 4) {
        // ================================================= softmax / tangent weights / epilogue (both CTAs) ========
        const int row = threadIdx.x - 128;                       // query row inside this CTA's half = TMEM lane
        const int prow = row + BR * (int)rank;                   // row inside the 256-row tile of the pair
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const float sl2 = prm.scale_log2, sc = prm.scale;
        const uint64_t sl2_2 = pack2(sl2, sl2), sc_2 = pack2(sc, sc);
        const uint32_t p_full = lead_bars + 8 * BAR_P_FULL, h_full = lead_bars + 8 * BAR_H_FULL;
        uint32_t c_s = 0, c_ts = 0, c_pv = 0;                    // uses of the S / tS barrier sets, pair-steps (PV_DONE)
        for (int it = list_begin; it < list_end; ++it) {
            if (sh->abort_flag) break;
            const aj_task task = prm.tasks[prm.pair_ids[it]];
            const int n = task.num_kv_tiles;
            const bool primal = (task.flags & AJ_TASK_PRIMAL_ONLY) != 0;
            float m_ref = M_UNSET;
            uint64_t l2[2] = {0ull, 0ull}, r2[2] = {0ull, 0ull};   // 4 partial sums each of l = sum P~ and r = sum H~
            RowCursor cur;
            cur.init(prm.k_begin, prm.k_end, prm.rows, task.range_begin, task.range_count, prow);
            const int np = (n + 1) >> 1;
            for (int p = 0; p < np; ++p, ++c_pv) {
                // columns of the two tiles this row may see: inside the entry's keys and row interval
                int valid[2];
                if (cur.pair_inside()) {
                    valid[0] = valid[1] = cur.pair();
                } else {
                    valid[0] = cur.tile();
                    valid[1] = 2 * p + 1 < n ? cur.tile() : 0;
                }
                // primal-only tasks alternate between the S columns (even pair-steps) and the tS columns (odd) as S buffer
                const bool alt = primal && (p & 1);
                const uint32_t tm_s = alt ? TM_TS : TM_S;
                wait(alt ? BAR_TS_FULL : BAR_S_FULL, (alt ? c_ts : c_s) & 1);
                tc_fence_after();
                uint32_t su[2][2][32];
                tmem_ld32(tmem + lane_base + tm_s, su[0][0]);
                tmem_ld32(tmem + lane_base + tm_s + 32, su[0][1]);
                tmem_ld32(tmem + lane_base + tm_s + 64, su[1][0]);
                tmem_ld32(tmem + lane_base + tm_s + 96, su[1][1]);
                tc_wait_ld(su[0][0], su[0][1]);
                tc_wait_ld(su[1][0], su[1][1]);
#pragma unroll
                for (int i = 0; i < 2; ++i)
                    if (valid[i] < BC) {
#pragma unroll
                        for (int c = 0; c < BC; ++c) if (c >= valid[i]) su[i][c >> 5][c & 31] = 0xff800000u;
                    }
                // P~ = exp2(S*s*log2e - m_ref); l += rowsum.  The bf16 pairs stay in registers for H~.
                uint32_t pk[2][32];
                uint64_t ls[2];                                   // this tile's contribution to l (committed once m_ref is settled)
                auto exp_tile = [&](int i, float mref) {
                    const uint64_t negm2 = pack2(-mref, -mref);
                    ls[0] = 0ull; ls[1] = 0ull;
#pragma unroll
                    for (int c = 0; c < BC / 2; ++c) {
                        const uint64_t x = ffma2(pack2(su[i][c >> 4][(2 * c) & 31], su[i][c >> 4][(2 * c + 1) & 31]), sl2_2, negm2);
                        float x0, x1;
                        unpack2(x, x0, x1);
                        const float p0 = ex2(x0), p1 = ex2(x1);
                        ls[c & 1] = fadd2(ls[c & 1], pack2(p0, p1));
                        pk[i][c] = pack_bf16(p0, p1);
                    }
                };
                float mx[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) mx[k] = __uint_as_float(su[0][0][k]);
#pragma unroll
                for (int c = 4; c < 2 * BC; ++c) mx[c & 3] = fmaxf(mx[c & 3], __uint_as_float(su[c >> 6][(c >> 5) & 1][c & 31]));
                const float cand = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * sl2;
                {
                    // Lazy reference max (PAPER.md:922-927 applied only when needed), once per pair-step: it moves only when
                    // the pair-step's max exceeds it by 2^8 (first pair-step of a task; later only for growing scores).
                    // A row whose reference is still unset has O = T = l = r = 0 exactly: it adopts the max with nothing
                    // to rescale.
                    const bool need = cand > m_ref + RESCALE_THRESHOLD;
                    if (__any_sync(0xffffffffu, need)) {
                        const bool fresh = m_ref == M_UNSET;
                        if (__any_sync(0xffffffffu, need && !fresh)) {
                            // e^{m - m_new} applied to O, T (= A + B), l, r; every MMA of the previous pair-step must be complete
                            wait(BAR_PV_DONE, (c_pv - 1) & 1);
                            tc_fence_after();
                            const float f = (need && !fresh) ? ex2(m_ref - cand) : 1.f;
                            const int ncols = primal ? 128 : 256;          // a primal-only task has no T
#pragma unroll 1
                            for (int cb = 0; cb < ncols; cb += 32) {
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
                }
                // Last pair-step of a primal-only task: S(p) only proves the MMAs of pair-step p - 2 complete (the pipe produced
                // it after them); the MMAs of p - 1 are waited for HERE, while those of p cannot have started (they need this
                // thread's P~), so that the epilogue's wait for pair-step p finds the barrier exactly one phase away.
                if (primal && p + 1 == np && np >= 2) wait(BAR_PV_DONE, (c_pv - 1) & 1);
                const uint32_t p_arrive = alt ? h_full : p_full;
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    // tile j1's exponentials must not be hoisted above tile j0's store and arrive (the P~ MMAs of j0 run
                    // under them): the reference passes through an opaque, ordered asm
                    float m_i = m_ref;
                    if (i == 1) {
                        // (ptxas would otherwise schedule all 128 MUFUs in front of the first tcgen05.st: tile j1's
                        // reference is made to depend on a shared-memory load that follows the arrive in program order)
                        uint32_t z;
                        asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(z) : "r"(smem_u32(&sh->abort_flag)) : "memory");
                        m_i = z ? M_UNSET : m_ref;
                    }
                    exp_tile(i, m_i);
                    l2[0] = fadd2(l2[0], ls[0]); l2[1] = fadd2(l2[1], ls[1]);
                    tmem_st32(tmem + lane_base + tm_s + i * BC, pk[i]);
                    tc_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(p_arrive + 8 * i);
                }
                if (primal) {                                    // no tS, no H~: the other buffer's S is next
                    if (alt) ++c_ts; else ++c_s;
                    continue;
                }
                // H~ = P~ o (s * tS); r += rowsum.  P~ is the bf16 value the MMAs see; masked columns
                // have P~ = 0, so H~ = 0.
                wait(BAR_TS_FULL, c_ts & 1);
                tc_fence_after();
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    uint32_t tu[2][32], hk[32];
                    tmem_ld32(tmem + lane_base + TM_TS + i * BC, tu[0]);
                    tmem_ld32(tmem + lane_base + TM_TS + i * BC + 32, tu[1]);
                    tc_wait_ld(tu[0], tu[1]);
#pragma unroll
                    for (int c = 0; c < BC / 2; ++c) {
                        const uint64_t tsc = fmul2(pack2(tu[c >> 4][(2 * c) & 31], tu[c >> 4][(2 * c + 1) & 31]), sc_2);
                        const uint64_t h = fmul2(pack2(pk[i][c] << 16, pk[i][c] & 0xffff0000u), tsc);
                        r2[c & 1] = fadd2(r2[c & 1], h);
                        float h0, h1;
                        unpack2(h, h0, h1);
                        hk[c] = pack_bf16(h0, h1);
                    }
                    tmem_st32(tmem + lane_base + TM_TS + i * BC, hk);
                    tc_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(h_full + 8 * i);
                }
                ++c_s;
                ++c_ts;
            }
            // ---- epilogue (Eq. 45) ----
            const bool store = prow < task.q_rows;
            const int64_t grow = task.q_begin + prow;
            __nv_bfloat16 *op = (__nv_bfloat16 *)prm.o.ptr + task.b * prm.o.stride_b + task.h * prm.o.stride_h + grow * prm.o.stride_n;
            __nv_bfloat16 *tp = prm.to.ptr ? (__nv_bfloat16 *)prm.to.ptr + task.b * prm.to.stride_b + task.h * prm.to.stride_h + grow * prm.to.stride_n : nullptr;
            if (n == 0) {                                         // no key: O = 0, tO = 0, lse = -inf (R9)
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = 0; c < D / 8; ++c) { ((uint4 *)op)[c] = z; if (tp) ((uint4 *)tp)[c] = z; }
                    if (prm.lse) prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = -INFINITY;
                    if (prm.tlse) prm.tlse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = 0.f;
                }
                continue;
            }
            // A parity wait is sound only if the barrier is known to be at most one phase away.  General task: tS of the last
            // pair-step was consumed, and the pipe produced it after the MMAs of the pair-step before.  Primal-only task:
            // the last pair-step waited for the one before it ahead of handing over its P~ (see there).
            wait(BAR_PV_DONE, (c_pv - 1) & 1);
            tc_fence_after();
            float la, lb, lc, ld, ra, rb, rc, rd;
            unpack2(l2[0], la, lb); unpack2(l2[1], lc, ld);
            unpack2(r2[0], ra, rb); unpack2(r2[1], rc, rd);
            const float l = (la + lb) + (lc + ld), r = (ra + rb) + (rc + rd);
            const float inv = l > 0.f ? 1.f / l : 0.f, rl = r * inv;   // l = 0: the row saw no key (O = 0, tO = 0, lse = -inf)
            if (primal) {
                // every tangent the task touches is zero: tO = 0 exactly (written only if the caller passed `to`)
#pragma unroll 1
                for (int cb = 0; cb < D; cb += 32) {
                    uint32_t ao[32];
                    tmem_ld32(tmem + lane_base + TM_O + cb, ao);
                    tc_wait_ld(ao);
                    if (store) {
#pragma unroll
                        for (int v4 = 0; v4 < 4; ++v4) {
                            uint32_t wo[4];
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int c = v4 * 8 + 2 * e;
                                wo[e] = pack_bf16(__uint_as_float(ao[c]) * inv, __uint_as_float(ao[c + 1]) * inv);
                            }
                            *(uint4 *)(op + cb + v4 * 8) = make_uint4(wo[0], wo[1], wo[2], wo[3]);
                            if (tp) *(uint4 *)(tp + cb + v4 * 8) = make_uint4(0, 0, 0, 0);
                        }
                    }
                }
            } else {
#pragma unroll 1
                for (int cb = 0; cb < D; cb += 32) {
                    uint32_t ao[32], at[32];
                    tmem_ld32(tmem + lane_base + TM_O + cb, ao);
                    tmem_ld32(tmem + lane_base + TM_T + cb, at);
                    tc_wait_ld(ao, at);
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
                            *(uint4 *)(tp + cb + v4 * 8) = make_uint4(wt[0], wt[1], wt[2], wt[3]);
                        }
                    }
                }
            }
            if (store && prm.lse)
                prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = l > 0.f ? (m_ref + log2f(l)) * 0.6931471805599453f : -INFINITY;
            // tangent of lse: sum_b p_ab tS_ab = r / l; a primal-only task has tS = 0 throughout
            if (store && prm.tlse)
                prm.tlse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = primal ? 0.f : rl;
            tc_fence_before();
        }
    }

    // Neither CTA may leave while the peer can still signal its barriers or the pair's MMAs write its TMEM.
    tc_fence_before();
    __syncthreads();
    cluster_arrive();
    cluster_wait();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    }
}

}  // namespace

size_t umma_pair_smem_bytes() { return SMEM_TOTAL; }

cudaError_t launch_umma_pair(const UmmaParams &prm, int num_pairs, cudaStream_t stream) {
    if (num_pairs <= 0) return cudaSuccess;
    static std::atomic<uint64_t> configured{0};
    if (cudaError_t e = ensure_dynamic_smem(attn_jvp_umma_pair_kernel, (int)SMEM_TOTAL, configured)) return e;
    attn_jvp_umma_pair_kernel<<<2 * num_pairs, NTHREADS, SMEM_TOTAL, stream>>>(prm);
    return cudaGetLastError();
}

}  // namespace aj
