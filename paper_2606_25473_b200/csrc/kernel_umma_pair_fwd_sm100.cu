// bf16 masked attention WITHOUT tangents for sm_100a on CTA pairs: the primal-only tasks of the forward.
//
// "The tangent of the clean context is zero" makes every clean x clean pair of a teacher-forcing call -- and
// every pair of the non-JVP stages and of the rollout's chunk-against-cached-prefix attention -- plain
// attention: S = Q K^T, O += P~ V (2 of the 6 contractions, Alg. 1 :913, :928-930).  In kernel_umma_pair_sm100.cu those
// pair-steps are bound by ONE softmax warp per scheduler, which serialises TMEM load -> 128-wide max -> 128 exponentials ->
// pack -> TMEM store (ncu: tensor pipe 47 %).  This kernel runs the same tasks with the softmax role doubled:
//   task / pair-step / operand staging as in the CTA-pair forward (256 query rows per SM pair, two 64-key tiles per step,
//   CTA c stages K(j_c) and the column half [64 c, 64 c + 64) of V(j0), V(j1); M256 N128 K16 MMAs)
//   TMEM (512 columns per CTA): O 128 | three S buffers of 128 (there is no tangent accumulator, so S is triple-buffered:
//   the MMA warp runs up to three pair-steps ahead of the softmax)
//   TWO softmax warpgroups (warps 4-7, 8-11; 12 warps per CTA) take ALTERNATE pair-steps, so that the exponentials of one
//   step overlap the load / max / store phases of the next.  A row's lazy reference max (PAPER.md:916-927 applied only when
//   the tile max exceeds it by 2^8) is handed from the warp that decided it for step g to its twin in the other warpgroup
//   through shared memory and a 64-thread named barrier; each warpgroup sums its own share of l and the two are combined
//   (rescaled to the final reference) in the epilogue.  The softmax warps run under a raised register budget (setmaxnreg:
//   208 registers, the producer / MMA / allocator warps give theirs back: 80), so all 128 scores of a pair-step come into
//   registers in ONE TMEM round trip and stay there across the reference-max decision (168 registers forced three round trips:
//   5.98 -> 5.66 ms on configs[1]'s mask); the branch holds no function call (PairWaiterInline), or ptxas would spill everything
//   live across it; tile j1 is handed to the MMA warp first.
//   All exponentials run on the MUFU pipe.  At d = 128 a tangent-free pair-step is 1024 clk of tensor work against
//   128 x 128 exponentials = 1024 clk of the 16-lane/clk MUFU pipe, so that pipe has no slack; moving every other column pair to
//   a polynomial on the FMA pipe was built and measured SLOWER (8.42 against 5.95 ms: the softmax warps are issue-bound, and
//   the polynomial costs ten instructions for the MUFU's one) and is not in the product.
// Roles per CTA: warp 0 TMA producer, warp 1 MMA issuer (leader CTA), warp 2 TMEM allocator (80 registers), warps 4-11 softmax /
// epilogue (208 registers).
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
using pairk::BC;
using pairk::PairWaiter;
using pairk::PairWaiterInline;
using pairk::RowCursor;
using pairk::Tile;
using pairk::TileCursor;

constexpr int BR = 128;                // query rows per CTA (UMMA M = 256 over the pair)
constexpr int D = 128;
constexpr int NSTAGE = 10;             // ring slots of 16 KB: {K of this CTA's tile} and {this CTA's half of V(j0), V(j1)} alternate
constexpr int NSBUF = 3;               // S buffers in TMEM
// Register budget per role (setmaxnreg, whole warpgroups: warps 0-3 / 4-7 / 8-11): 128 x 80 + 256 x 208 = 63,488 of the SM's 65,536.
constexpr int REG_MISC = 80, REG_ROLE = 208;
constexpr uint32_t Q_BYTES = BR * D * 2;           // 32 KB
constexpr uint32_t QHALF_BYTES = BR * 64 * 2;      // 16 KB: one 64-column swizzle block of Q
constexpr uint32_t BLK_BYTES = BC * 64 * 2;        // 8 KB: 64 keys x 64 columns, 128-byte swizzled rows
constexpr uint32_t SLOT_BYTES = 2 * BLK_BYTES;     // 16 KB
constexpr uint32_t SMEM_TILES = Q_BYTES + NSTAGE * SLOT_BYTES;      // 192 KB
constexpr uint32_t SMEM_TOTAL = SMEM_TILES + 1024 /*align*/ + 4096 /*struct Shared*/;
constexpr int NTHREADS = 384;

constexpr uint32_t TM_O = 0, TM_S = 128;           // S buffer b at TM_S + 128 b; P~(j_i) over the first 32 columns of its tile's 64
constexpr float RESCALE_THRESHOLD = 8.0f;          // log2 units
constexpr float M_UNSET = -1.0e30f;

enum {
    BAR_Q_FULL = 0,                         // leader: Q of both CTAs landed
    BAR_Q_EMPTY,                            // both: every S MMA of the task is complete
    BAR_KV_FULL,                            // leader: ring slot filled in both CTAs
    BAR_KV_EMPTY = BAR_KV_FULL + NSTAGE,    // both
    BAR_S_FULL = BAR_KV_EMPTY + NSTAGE,     // both, x NSBUF
    BAR_P_FULL = BAR_S_FULL + NSBUF,        // leader, x NSBUF x 2 tiles: P~ stored by the step's warpgroup in both CTAs
    BAR_PV_DONE = BAR_P_FULL + 2 * NSBUF,   // both, x NSBUF: every MMA up to and including the step's P~ V is complete
    NUM_BARS = BAR_PV_DONE + NSBUF
};

constexpr uint32_t make_idesc(int n, bool b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}
constexpr uint32_t IDESC_QK = make_idesc(2 * BC, false);
constexpr uint32_t IDESC_PV = make_idesc(D, true);
constexpr uint32_t DESC_HI = desc_hi(1024);
constexpr uint32_t LBO_CANON = desc_lo_lbo(16);

struct Shared {
    uint64_t bars[NUM_BARS];
    uint32_t tmem_base;
    int abort_flag;
    float mref[2][BR];          // reference max handed from the warp of step g to its twin for step g + 1 (slot g & 1)
    float fin_m[2][BR];         // epilogue: each warpgroup's reference max and share of l
    float fin_l[2][BR];
};
static_assert(sizeof(Shared) <= 4096, "struct Shared outgrew its reservation");

__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
attn_fwd_umma_pair_kernel(const __grid_constant__ UmmaParams prm) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;
    Shared *sh = reinterpret_cast<Shared *>(smem_raw + (tiles - raw) + SMEM_TILES);
    const uint32_t sQ = tiles, sRing = tiles + Q_BYTES;
    const uint32_t bars = smem_u32(sh->bars);
    const PairWaiter wait{bars, &sh->abort_flag, prm.counters + 2, 400};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const uint32_t lead_bars = mapa(bars, 0);
    const int pair = blockIdx.x >> 1;
    const int list_begin = prm.pair_off[pair], list_end = prm.pair_off[pair + 1];

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * BAR_Q_FULL, 1);
        mbar_init(bars + 8 * BAR_Q_EMPTY, 1);
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bars + 8 * (BAR_KV_FULL + i), 1); mbar_init(bars + 8 * (BAR_KV_EMPTY + i), 1); }
        for (int b = 0; b < NSBUF; ++b) {
            mbar_init(bars + 8 * (BAR_S_FULL + b), 1);
            mbar_init(bars + 8 * (BAR_P_FULL + 2 * b), 8);       // the step's warpgroup: 4 warps in each CTA
            mbar_init(bars + 8 * (BAR_P_FULL + 2 * b + 1), 8);
            mbar_init(bars + 8 * (BAR_PV_DONE + b), 1);
        }
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
    cluster_arrive();
    cluster_wait();
    tc_fence_after();
    const uint32_t tmem = sh->tmem_base;

    // Each branch below is dominated by its own setmaxnreg, which is what lets ptxas allocate it against that budget; the softmax
    // branch contains no function call (PairWaiterInline), or everything live across the call would be spilled.
    if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REG_MISC));
    if (warp == 0) {
        // ================================================= TMA producer (both CTAs) ================================
        if (lane == 0) {
            prefetch_tmap(&prm.tm_q); prefetch_tmap(&prm.tm_k); prefetch_tmap(&prm.tm_v);
            uint32_t ring = 0, nq = 0;
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task task = prm.tasks[prm.pair_ids[it]];
                const int n = task.num_kv_tiles;
                if (n == 0 || sh->abort_flag) continue;
                wait(BAR_Q_EMPTY, (nq & 1) ^ 1);
                const uint32_t qfull = lead_bars + 8 * BAR_Q_FULL;
                if (rank == 0) mbar_expect_tx(bars + 8 * BAR_Q_FULL, 2 * Q_BYTES);
                const int qrow = task.q_begin + BR * (int)rank;
                tma_load_4d_pair(sQ, &prm.tm_q, qfull, 0, qrow, task.h, task.b);
                tma_load_4d_pair(sQ + QHALF_BYTES, &prm.tm_q, qfull, 64, qrow, task.h, task.b);
                ++nq;
                TileCursor cur;
                cur.init(prm.k_begin, prm.k_end, task.range_begin, task.range_count);
                const int np = (n + 1) >> 1;
                for (int p = 0; p < np; ++p) {
                    const Tile t0 = cur.get();
                    cur.next();
                    Tile t1 = t0;                          // odd tail: the second tile is a fully masked copy of the first
                    if (2 * p + 1 < n) { t1 = cur.get(); cur.next(); }
                    {   // K of this CTA's tile: [K h0 | K h1]
                        const uint32_t slot = ring % NSTAGE;
                        wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                        const uint32_t dst = sRing + slot * SLOT_BYTES, full = lead_bars + 8 * (BAR_KV_FULL + slot);
                        if (rank == 0) mbar_expect_tx(bars + 8 * (BAR_KV_FULL + slot), 2 * SLOT_BYTES);
                        const int row = rank ? t1.key_row : t0.key_row;
                        tma_load_4d_pair(dst, &prm.tm_k, full, 0, row, task.h, task.b);
                        tma_load_4d_pair(dst + BLK_BYTES, &prm.tm_k, full, 64, row, task.h, task.b);
                        ++ring;
                    }
                    {   // this CTA's column half of V of both tiles: [V(j0) | V(j1)]
                        const uint32_t slot = ring % NSTAGE;
                        wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                        const uint32_t dst = sRing + slot * SLOT_BYTES, full = lead_bars + 8 * (BAR_KV_FULL + slot);
                        if (rank == 0) mbar_expect_tx(bars + 8 * (BAR_KV_FULL + slot), 2 * SLOT_BYTES);
                        const int col = 64 * (int)rank;
                        tma_load_4d_pair(dst, &prm.tm_v, full, col, t0.key_row, task.h, task.b);
                        tma_load_4d_pair(dst + BLK_BYTES, &prm.tm_v, full, col, t1.key_row, task.h, task.b);
                        ++ring;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ================================================= MMA issuer (leader CTA) ==================================
        if (rank == 0) {
            const bool leader = elect_one();
            const uint32_t q_lo = ((sQ >> 4) & 0x3FFF) | LBO_CANON;
            uint32_t ring = 0, nq = 0, g0 = 0;            // ring items before this task; tasks; pair-steps before this task
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task &tk = prm.tasks[prm.pair_ids[it]];
                const int n = (int)warp_uniform((uint32_t)tk.num_kv_tiles | (sh->abort_flag ? 0x80000000u : 0u));
                if (n <= 0) continue;
                wait(BAR_Q_FULL, nq & 1);
                ++nq;
                tc_fence_after();
                const int np = (n + 1) >> 1;
                const uint32_t base = ring;               // ring items: K(p) = base + 2p, V(p) = base + 2p + 1
                ring += 2 * (uint32_t)np;
                auto issue_S = [&](int p) {
                    const uint32_t item = base + 2 * (uint32_t)p, slot = item % NSTAGE, g = g0 + (uint32_t)p, buf = g % NSBUF;
                    wait(BAR_KV_FULL + slot, (item / NSTAGE) & 1);
                    tc_fence_after();
                    const uint32_t k_lo = (((sRing + slot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
                    if (leader) {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {   // [S(j0) | S(j1)] = Q [K(j0) ; K(j1)]^T
                            const uint32_t qoff = ((ks >> 2) * QHALF_BYTES + (ks & 3) * 32) >> 4;
                            const uint32_t koff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                            mma_ss_pair(tmem + TM_S + 128 * buf, q_lo + qoff, DESC_HI, k_lo + koff, DESC_HI, IDESC_QK, ks > 0);
                        }
                        tc_commit_pair(bars + 8 * (BAR_S_FULL + buf), 3);
                        tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + slot), 3);
                        if (p + 1 == np) tc_commit_pair(bars + 8 * BAR_Q_EMPTY, 3);
                    }
                    __syncwarp();
                };
                for (int p = 0; p < NSBUF && p < np; ++p) issue_S(p);
                for (int p = 0; p < np; ++p) {
                    const uint32_t item = base + 2 * (uint32_t)p + 1, vslot = item % NSTAGE, g = g0 + (uint32_t)p, buf = g % NSBUF;
                    wait(BAR_KV_FULL + vslot, (item / NSTAGE) & 1);
                    const uint32_t v_lo = (((sRing + vslot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
#pragma unroll
                    for (int ii = 0; ii < 2; ++ii) {
                        const int i = 1 - ii;                        // the softmax hands over tile j1 first (it keeps S(j1) in registers)
                        const uint32_t vi_lo = v_lo + ((i * BLK_BYTES) >> 4);
                        const uint32_t tP = tmem + TM_S + 128 * buf + i * BC;
                        const uint32_t acc = (p > 0 || ii > 0) ? 1u : 0u;
                        wait(BAR_P_FULL + 2 * buf + i, (g / NSBUF) & 1);
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
                        tc_commit_pair(bars + 8 * (BAR_PV_DONE + buf), 3);
                    }
                    __syncwarp();
                    if (p + NSBUF < np) issue_S(p + NSBUF);          // overwrites P~(p): the pipe executes in order
                }
                g0 += (uint32_t)np;
            }
        }
    }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_ROLE));
        const PairWaiterInline wait{bars, &sh->abort_flag, prm.counters + 2, 400};
        // ================================================= softmax / epilogue (both CTAs, two warpgroups) ==========
        const int wg = (warp - 4) >> 2;                          // takes the pair-steps whose global index has this parity
        const int q4 = warp & 3;                                 // lane quarter of TMEM = warp index inside the warpgroup
        const int row = (threadIdx.x - 128) & (BR - 1);          // query row inside this CTA's half = TMEM lane
        const int prow = row + BR * (int)rank;
        const uint32_t lane_base = (uint32_t)(q4 * 32) << 16;
        const float sl2 = prm.scale_log2;
        const uint64_t sl2_2 = pack2(sl2, sl2);
        uint32_t g0 = 0;                                         // pair-steps before this task
        for (int it = list_begin; it < list_end; ++it) {
            if (sh->abort_flag) break;
            const aj_task task = prm.tasks[prm.pair_ids[it]];
            const int n = task.num_kv_tiles;
            float m_ref = M_UNSET;
            uint64_t l2[2] = {0ull, 0ull};                       // 4 partial sums of this warpgroup's share of l = sum P~
            RowCursor cur;
            cur.init(prm.k_begin, prm.k_end, prm.rows, task.range_begin, task.range_count, prow);
            const int np = (n + 1) >> 1;
            // This warpgroup's pair-steps are those whose global index g0 + p has its parity: p = first, first + 2, ...  The loop visits
            // only them (the bookkeeping of a visited step is ~50 scalar instructions with half a dozen branches, ~300 clk on a warp
            // that has nothing else to issue: visiting the twin's steps as well cost 600 clk per own step); the twin's step that follows
            // is consumed from the cursor together with the own one.  S buffer and barrier phase advance by two steps at a time.
            const int first = (int)((g0 ^ (uint32_t)wg) & 1u);
            auto skip_step = [&](int q) {                        // consume pair-step q of the stream without using it
                if (cur.pair_inside()) cur.pair();
                else { cur.tile(); if (2 * q + 1 < n) cur.tile(); }
            };
            if (first == 1 && np > 0) skip_step(0);
            uint32_t buf = (g0 + (uint32_t)first) % NSBUF, sph = ((g0 + (uint32_t)first) / NSBUF) & 1;
            for (int p = first; p < np; p += 2) {
                const uint32_t g = g0 + (uint32_t)p;
                int valid[2];
                if (cur.rem >= 4 * BC) {                         // the own step and the twin's next one lie inside the current entry
                    valid[0] = valid[1] = cur.sees ? BC : 0;
                    cur.rem -= 4 * BC;
                    if (cur.rem <= 0) cur.advance();
                } else {
                    if (cur.pair_inside()) {
                        valid[0] = valid[1] = cur.pair();
                    } else {
                        valid[0] = cur.tile();
                        valid[1] = 2 * p + 1 < n ? cur.tile() : 0;
                    }
                    if (p + 1 < np) skip_step(p + 1);
                }
                const uint32_t tS = tmem + lane_base + TM_S + 128 * buf;
                wait(BAR_S_FULL + buf, sph);
                tc_fence_after();
                // ---- pass 1: the pair-step's row max over the columns this row may see.  All 128 scores of the
                // step come into registers in ONE TMEM round trip (four loads in flight) and stay there for pass 2.
                float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
                uint32_t s0a[32], s0b[32], s1a[32], s1b[32];
                tmem_ld32(tS, s0a);
                tmem_ld32(tS + 32, s0b);
                tmem_ld32(tS + 64, s1a);
                tmem_ld32(tS + 96, s1b);
                // the twin's reference max of step g - 1 is fetched under the TMEM round trip (the twin decided it long ago)
                float m_prev = m_ref;
                if (p > 0) {
                    named_bar_sync(1 + 2 * q4 + (int)((g - 1) & 1), 64);
                    m_prev = sh->mref[(g - 1) & 1][row];
                }
                tc_wait_ld(s0a, s0b);
                tc_wait_ld(s1a, s1b);
                if (valid[0] < BC) {                            // outside the entry's keys / row interval: S = -inf (P~ = 0)
#pragma unroll
                    for (int c = 0; c < 32; ++c) { if (c >= valid[0]) s0a[c] = 0xff800000u; if (c + 32 >= valid[0]) s0b[c] = 0xff800000u; }
                }
                if (valid[1] < BC) {
#pragma unroll
                    for (int c = 0; c < 32; ++c) { if (c >= valid[1]) s1a[c] = 0xff800000u; if (c + 32 >= valid[1]) s1b[c] = 0xff800000u; }
                }
#pragma unroll
                for (int c = 0; c < 32; c += 2) {                // 3-input max (FMNMX3): 64 instead of 128 instructions on the ALU pipe
                    mx[0] = max3(mx[0], __uint_as_float(s0a[c]), __uint_as_float(s0a[c + 1]));
                    mx[1] = max3(mx[1], __uint_as_float(s0b[c]), __uint_as_float(s0b[c + 1]));
                    mx[2] = max3(mx[2], __uint_as_float(s1a[c]), __uint_as_float(s1a[c + 1]));
                    mx[3] = max3(mx[3], __uint_as_float(s1b[c]), __uint_as_float(s1b[c + 1]));
                }
                const float cand = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * sl2;
                // ---- the reference max: taken over from the twin warp (step g - 1), moved only if this step's max exceeds it by 2^8
                if (p > 0) {
                    if (m_prev != m_ref) {                       // the twin moved it: this warpgroup's share of l follows
                        const float f = m_ref == M_UNSET ? 0.f : ex2(m_ref - m_prev);
                        const uint64_t f2 = pack2(f, f);
                        l2[0] = fmul2(l2[0], f2); l2[1] = fmul2(l2[1], f2);
                        m_ref = m_prev;
                    }
                }
                {
                    const bool need = cand > m_ref + RESCALE_THRESHOLD;
                    if (__any_sync(0xffffffffu, need)) {
                        const bool fresh = m_ref == M_UNSET;         // first pair-step of the task: O = l = 0, nothing to rescale
                        if (__any_sync(0xffffffffu, need && !fresh)) {
                            // e^{m - m_new} applied to O and l; every MMA of the steps before must be complete.
                            // S(g) complete proves P~ V of step g - 3 complete, so this barrier is at most one phase away.
                            wait(BAR_PV_DONE + (g - 1) % NSBUF, ((g - 1) / NSBUF) & 1);
                            tc_fence_after();
                            const float f = (need && !fresh) ? ex2(m_ref - cand) : 1.f;
#pragma unroll 1
                            for (int cb = 0; cb < D; cb += 32) {
                                uint32_t a[32];
                                tmem_ld32(tmem + lane_base + TM_O + cb, a);
                                tc_wait_ld(a);
#pragma unroll
                                for (int c = 0; c < 32; ++c) a[c] = __float_as_uint(__uint_as_float(a[c]) * f);
                                tmem_st32(tmem + lane_base + TM_O + cb, a);
                            }
                            tc_wait_st();
                            const uint64_t f2 = pack2(f, f);
                            l2[0] = fmul2(l2[0], f2); l2[1] = fmul2(l2[1], f2);
                        }
                        if (need) m_ref = cand;
                    }
                }
                if (p + 1 < np) {                                // hand the reference to the twin warp for step g + 1
                    sh->mref[g & 1][row] = m_ref;
                    named_bar_arrive(1 + 2 * q4 + (int)(g & 1), 64);
                }
                // ---- pass 2: P~ = exp2(S s log2e - m_ref); l += rowsum; bf16 P~ over the tile's first 32 columns.
                // Masked columns hold -inf: exp2(-inf) = 0 exactly.
                const uint64_t negm2 = pack2(-m_ref, -m_ref);
                auto exp_tile = [&](int i, const uint32_t (&a)[32], const uint32_t (&b)[32]) {
                    uint32_t pk[32];
#pragma unroll
                    for (int c = 0; c < 64; c += 2) {
                        const uint32_t u0 = c < 32 ? a[c & 31] : b[c & 31], u1 = c < 32 ? a[(c + 1) & 31] : b[(c + 1) & 31];
                        const uint64_t x = ffma2(pack2(u0, u1), sl2_2, negm2);
                        float x0, x1;
                        unpack2(x, x0, x1);
                        const uint64_t e = pack2(ex2(x0), ex2(x1));
                        l2[(c >> 1) & 1] = fadd2(l2[(c >> 1) & 1], e);
                        float p0, p1;
                        unpack2(e, p0, p1);
                        pk[c >> 1] = pack_bf16(p0, p1);
                    }
                    tmem_st32(tS + 64 * i, pk);
                    tc_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(lead_bars + 8 * (BAR_P_FULL + 2 * buf + i));
                };
                exp_tile(1, s1a, s1b);                              // tile j1 is handed to the MMA warp first
                exp_tile(0, s0a, s0b);
                buf += 2;                                           // two pair-steps on: S buffer (g + 2) % 3 and its barrier phase
                if (buf >= NSBUF) { buf -= NSBUF; sph ^= 1; }
            }
            // ---- epilogue: O / l, lse = m + log l; each warpgroup writes one 64-column half ----
            const bool store = prow < task.q_rows;
            const int64_t grow = task.q_begin + prow;
            __nv_bfloat16 *op = (__nv_bfloat16 *)prm.o.ptr + task.b * prm.o.stride_b + task.h * prm.o.stride_h + grow * prm.o.stride_n;
            __nv_bfloat16 *tp = prm.to.ptr ? (__nv_bfloat16 *)prm.to.ptr + task.b * prm.to.stride_b + task.h * prm.to.stride_h + grow * prm.to.stride_n : nullptr;
            const int64_t lrow = ((int64_t)task.b * prm.H + task.h) * prm.Nq + grow;
            if (n == 0) {                                         // no key: O = 0, tO = 0, lse = -inf (R9)
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = 8 * wg; c < 8 * wg + 8; ++c) { ((uint4 *)op)[c] = z; if (tp) ((uint4 *)tp)[c] = z; }
                    if (wg == 0 && prm.lse) prm.lse[lrow] = -INFINITY;
                    if (wg == 0 && prm.tlse) prm.tlse[lrow] = 0.f;
                }
                continue;
            }
            {
                float la, lb, lc, ld;
                unpack2(l2[0], la, lb); unpack2(l2[1], lc, ld);
                sh->fin_m[wg][row] = m_ref;
                sh->fin_l[wg][row] = (la + lb) + (lc + ld);
            }
            named_bar_sync(9, 256);                               // both warpgroups have handed over their last P~ and their sums
            const float m_a = sh->fin_m[0][row], m_b = sh->fin_m[1][row];
            const float m_fin = fmaxf(m_a, m_b);                  // the reference only ever grows; the staler side is rescaled to it
            const float l = sh->fin_l[0][row] * (m_a == M_UNSET ? 0.f : ex2(m_a - m_fin)) + sh->fin_l[1][row] * (m_b == M_UNSET ? 0.f : ex2(m_b - m_fin));
            // The warpgroup of the last pair-step saw S of that step, which the in-order pipe produced after P~ V of the step three
            // before: with the named barrier above both warpgroups know that this buffer's barrier is at most one phase away.
            {
                const uint32_t gl = g0 + (uint32_t)np - 1;
                wait(BAR_PV_DONE + gl % NSBUF, (gl / NSBUF) & 1);
                tc_fence_after();
            }
            const float inv = l > 0.f ? 1.f / l : 0.f;            // l = 0: the row saw no key (O = 0, lse = -inf)
#pragma unroll 1
            for (int cb = 64 * wg; cb < 64 * wg + 64; cb += 32) {
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
                        if (tp) *(uint4 *)(tp + cb + v4 * 8) = make_uint4(0, 0, 0, 0);     // every tangent the task touches is zero
                    }
                }
            }
            if (store && wg == 0) {
                if (prm.lse) prm.lse[lrow] = l > 0.f ? (m_fin + log2f(l)) * 0.6931471805599453f : -INFINITY;
                if (prm.tlse) prm.tlse[lrow] = 0.f;
            }
            tc_fence_before();
            named_bar_sync(10, 256);         // O and the hand-over slots are free only when both warpgroups are done
            g0 += (uint32_t)np;
        }
    }

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

cudaError_t launch_umma_pair_fwd(const UmmaParams &prm, int num_pairs, cudaStream_t stream) {
    if (num_pairs <= 0) return cudaSuccess;
    static std::atomic<uint64_t> configured{0};
    if (cudaError_t e = ensure_dynamic_smem(attn_fwd_umma_pair_kernel, (int)SMEM_TOTAL, configured)) return e;
    attn_fwd_umma_pair_kernel<<<2 * num_pairs, NTHREADS, SMEM_TOTAL, stream>>>(prm);
    return cudaGetLastError();
}

}  // namespace aj
