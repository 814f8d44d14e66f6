// bf16 primal backward of masked attention for sm_100a on CTA PAIRS: TMA -> shared-memory ring ->
// tcgen05.mma.cta_group::2 (M = 256) with TMEM accumulators.  Same formulas as kernel_simt_bwd.cu (the VJP of Eq. 42,
// PAPER.md:842-844):
//     p_ab = exp(s <q_a, k_b> - lse_a),  dP_ab = <dO_a, v_b>,  dS_ab = p_ab (dP_ab - delta_a),  delta_a = <dO_a, O_a>
//     dQ_a = s sum_b dS_ab k_b ;   dK_b = s sum_a dS_ab q_a ;   dV_b = sum_a p_ab dO_a
// Two passes of ONE kernel (the same computation with the roles swapped), re-tiled like the forward CTA-pair kernel
// (kernel_umma_pair_sm100.cu) so that every shared-memory-operand MMA has N = 128 and the two SMs share the stream:
//   task      = 256 STATIONARY rows of one (b, h) on the global 256-row grid (packed tiling): CTA c owns rows [128 c, 128 c + 128)
//   pair-step = TWO 64-row STREAMED tiles j0, j1 of the task's stream (CTA c stages tile j_c for the K-major operands and
//               the column half [64 c, 64 c + 64) of both tiles for the MN-major operands)
//     [X(j0) | X(j1)] = A1 [B1(j0) ; B1(j1)]^T,   [Y(j0) | Y(j1)] = A2 [B2(j0) ; B2(j1)]^T        2 x 8 x (M256 N128 K16)
//     W = exp2(X s log2e - lse log2e),   Z = W o (Y - delta)       two exp / dS warpgroups, 32 of a tile's 64 columns each,
//                                                                    tile j0 first; thread = stationary row = TMEM lane
//     per tile: acc1 += Z B1  (and acc2 += W B2)                    4 (+ 4) x (M256 N128 K16), A = bf16 Z / W in TMEM
//   dQ:                    attn_bwd_dq_pair_kernel below (tile ping-pong; stationary = query rows, Q and dO rows as bf16 A
//                          operands in TMEM).  A pair-step form of it used to be the KEYS = false instantiation of this
//                          template; it was measured slower and has been removed.
//   KEYS = true (dK, dV):  stationary = keys (A1 = K, A2 = V in shared memory), streamed = query rows (B1 = Q, B2 = dO):
//                          X = S^T, Y = dP^T, acc1 = dK / s, acc2 = dV; lse and delta belong to the COLUMNS, and they are
//                          folded INTO the two contractions: one extra K step (16 of the bf16 K dimension) multiplies a
//                          constant block of ones (A) with 16 extra columns per streamed row (B) that the delta kernel
//                          wrote: -lse/s (resp. -delta) split into bf16 hi + lo, so that the tensor pipe delivers
//                          X = <k, q> - lse/s and Y = <v, dO> - delta and the exp / dS warps read nothing per column
//                          (a shared-memory copy of lse / delta read by every thread cost 41 % of the shared-memory port
//                          and doubled the role's instruction count).  Tasks come from the transposed mask.
// S and dP are computed in both passes (7 contractions for the minimal 5): a single pass would need dK, dV, S^T, dP^T and a
// 128-column dQ partial = 640 TMEM columns and a cross-CTA reduction of dQ; DESIGN.md section 6d.
// TMEM (512 columns per CTA):  acc1 128 | acc2 128 (KEYS) or bf16 A1 64 + A2 64 (dQ pass) | X(j0) X(j1) 128 | Y(j0) Y(j1) 128;
// bf16 W / Z of a tile's streamed rows [32 h, 32 h + 32) overwrite columns [32 h, 32 h + 16) of the tile's X / Y.  X / Y are single-buffered; as in the forward the overlap
// comes from the issue order on the in-order tensor pipe:
//   KEYS:  W(j0) B2, W(j1) B2, X(p+1) [overwrites W], Z(j0) B1, Z(j1) B1, Y(p+1) [overwrites Z]
//   dQ:    X(p+1) [once the exp warps have LOADED X(p): X_FREE], Z(j0) B1, Z(j1) B1, Y(p+1)
// Roles per CTA (12 warps): warp 0 TMA producer, warp 1 MMA issuer (leader CTA), warp 2 TMEM allocator, warps 4-7 / 8-11
// exp / dS / epilogue warpgroup of tile j0 / j1.  Tasks are assigned to the pairs by the host (assign_workers), head-major.
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
using pairk::RowCursor;
using pairk::Tile;
using pairk::TileCursor;

constexpr int BR = 128;                // stationary rows per CTA (UMMA M = 256 over the pair)
constexpr int D = 128;
constexpr uint32_t A_BYTES = BR * D * 2;           // 32 KB
constexpr uint32_t AHALF_BYTES = BR * 64 * 2;      // one 64-column swizzle block of a stationary operand: 16 KB
constexpr uint32_t BLK_BYTES = BC * 64 * 2;        // 8 KB: 64 streamed rows x 64 columns, 128-byte swizzled rows
constexpr uint32_t SLOT_BYTES = 4 * BLK_BYTES;     // 32 KB
// KEYS: the K-augmentation operands.  A row of an aug array is 16 bf16 = 32 B: [h/2, l/2, 0 x 6, h/2, l/2, 0 x 6] with
// h + l = the folded value (both 16-byte halves alike, so no swizzle pattern can matter); the constant A block is 128 rows of
// [1, 1, 0 x 6, 1, 1, 0 x 6].  Both are read through K-major descriptors of the 32-byte-swizzle kind: rows 32 B apart, 8-row
// groups 256 B apart.
constexpr uint32_t AUG_TILE_BYTES = BC * 32;       // 2 KB: 64 streamed rows
constexpr uint32_t AUG_STAGE_BYTES = 2 * AUG_TILE_BYTES;   // q-aug and dO-aug of this CTA's tile
constexpr int AUG_STAGES = 2;                      // one per ring slot that can hold a {B1, B2} tile (slots 0 and 2 of 4)
constexpr uint32_t ONES_BYTES = BR * 32;           // 4 KB
constexpr int NTHREADS = 384;

template <bool KEYS> struct Cfg {
    static constexpr int NSTAGE = KEYS ? 4 : 6;                          // ring slots of 32 KB
    static constexpr uint32_t A_SMEM = KEYS ? 2 * A_BYTES : 0;           // stationary operands in shared memory (KEYS only)
    static constexpr uint32_t AUG_SMEM = KEYS ? AUG_STAGES * AUG_STAGE_BYTES + ONES_BYTES : 0;
    static constexpr uint32_t SMEM_TILES = A_SMEM + NSTAGE * SLOT_BYTES + AUG_SMEM;
    static constexpr uint32_t SMEM_TOTAL = SMEM_TILES + 1024 /*align*/ + 512 /*barriers*/;
};

constexpr uint32_t TM_ACC1 = 0, TM_ACC2 = 128, TM_A1 = 128, TM_A2 = 192, TM_X = 256, TM_Y = 384;

constexpr int MAX_STAGE = 6;
enum {
    BAR_A_FULL = 0,                         // leader: KEYS: A1, A2 of both CTAs landed (transaction bytes); dQ: 16 warps stored their rows
    BAR_A_EMPTY,                            // both: every X / Y MMA of the task is complete (KEYS)
    BAR_KV_FULL,                            // leader: ring slot filled in both CTAs
    BAR_KV_EMPTY = BAR_KV_FULL + MAX_STAGE, // both: the MMAs reading the slot are complete
    BAR_X_FULL = BAR_KV_EMPTY + MAX_STAGE,  // both
    BAR_Y_FULL,                             // both
    BAR_X_FREE,                             // leader: all 16 exp / dS warps of the pair have loaded X of the pair-step (dQ pass)
    BAR_W_FULL,                             // leader, x2 (tile): W stored by the tile's warpgroup in both CTAs (KEYS)
    BAR_Z_FULL = BAR_W_FULL + 2,            // leader, x2
    BAR_ACC_DONE = BAR_Z_FULL + 2,          // both: every MMA into acc1 / acc2 of the pair-step is complete
    NUM_BARS
};

// Instruction descriptor, kind::f16: D fp32, A and B bf16, N >> 3 at bit 17, M >> 4 at bit 24 (M = 256 over the pair).
constexpr uint32_t make_idesc(int n, bool b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}
constexpr uint32_t IDESC_XY = make_idesc(2 * BC, false);   // 256 x 128 x 16, B K-major (64 streamed rows per CTA)
constexpr uint32_t IDESC_ACC = make_idesc(D, true);        // 256 x 128 x 16, A from TMEM, B MN-major (64 columns per CTA)
constexpr uint32_t DESC_HI = desc_hi(1024);                // 8-row groups are 1024 B apart
constexpr uint32_t LBO_CANON = desc_lo_lbo(16);            // single 64-column block per operand: LBO unused
constexpr uint32_t DESC_HI_SW32 = ((256u >> 4) & 0x3FFF) | (1u << 14) | (6u << 29);   // 32-byte swizzle kind, 8-row groups 256 B apart

struct Shared {
    uint64_t bars[NUM_BARS];
    uint32_t tmem_base;
    int abort_flag;
};
static_assert(sizeof(Shared) <= 512, "struct Shared outgrew its reservation");

// 2-D TMA load (rows of an aug array) whose completion bytes go to a barrier of either CTA of the pair
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap *map, uint32_t cluster_bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(cluster_bar), "r"(c0), "r"(c1) : "memory");
}

template <bool KEYS>   // only KEYS = true exists (the dQ pass has its own kernel below); the parameter keeps the kernel's name
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
attn_bwd_umma_pair_kernel(const __grid_constant__ BwdPairParams prm) {
    static_assert(KEYS, "the pair-step form of the dQ pass was removed (measured slower: DESIGN.md 6d); dQ runs attn_bwd_dq_pair_kernel");
    using C = Cfg<KEYS>;
    constexpr int NSTAGE = C::NSTAGE;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;       // 1024-byte alignment for the 128-byte swizzle
    Shared *sh = reinterpret_cast<Shared *>(smem_raw + (tiles - raw) + C::SMEM_TILES);
    const uint32_t sA1 = tiles, sA2 = tiles + A_BYTES, sRing = tiles + C::A_SMEM, sAug = sRing + NSTAGE * SLOT_BYTES;
    const uint32_t sOnes = sAug + AUG_STAGES * AUG_STAGE_BYTES;
    const uint32_t bars = smem_u32(sh->bars);
    const PairWaiter wait{bars, &sh->abort_flag, prm.err, 300};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();              // 0 = leader (issues the MMAs, owns the "full" barriers)
    const uint32_t lead_bars = mapa(bars, 0);
    const int pair = blockIdx.x >> 1;
    const int list_begin = prm.pair_off[pair], list_end = prm.pair_off[pair + 1];

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * BAR_A_FULL, 1);
        mbar_init(bars + 8 * BAR_A_EMPTY, 1);
        for (int i = 0; i < MAX_STAGE; ++i) { mbar_init(bars + 8 * (BAR_KV_FULL + i), 1); mbar_init(bars + 8 * (BAR_KV_EMPTY + i), 1); }
        mbar_init(bars + 8 * BAR_X_FULL, 1);
        mbar_init(bars + 8 * BAR_Y_FULL, 1);
        mbar_init(bars + 8 * BAR_X_FREE, 16);
        for (int i = 0; i < 2; ++i) {
            mbar_init(bars + 8 * (BAR_W_FULL + i), 16);   // all 8 exp / dS warps of each CTA (32 of the tile's columns per warpgroup)
            mbar_init(bars + 8 * (BAR_Z_FULL + i), 16);
        }
        mbar_init(bars + 8 * BAR_ACC_DONE, 1);
        sh->abort_flag = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (threadIdx.x >= 128 && threadIdx.x < 128 + BR) {
        // the constant A operand of the augmentation step: row r = [1, 1, 0 x 6, 1, 1, 0 x 6] (bf16 1.0 = 0x3f80)
        uint8_t *ones = smem_raw + (tiles - raw) + C::A_SMEM + NSTAGE * SLOT_BYTES + AUG_STAGES * AUG_STAGE_BYTES + (threadIdx.x - 128) * 32;
        reinterpret_cast<uint4 *>(ones)[0] = make_uint4(0x3f803f80u, 0u, 0u, 0u);
        reinterpret_cast<uint4 *>(ones)[1] = make_uint4(0x3f803f80u, 0u, 0u, 0u);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // read by the tensor pipe (async proxy)
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
            prefetch_tmap(&prm.tm_b1); prefetch_tmap(&prm.tm_b2);
            prefetch_tmap(&prm.tm_a1); prefetch_tmap(&prm.tm_a2); prefetch_tmap(&prm.tm_aug1); prefetch_tmap(&prm.tm_aug2);
            uint32_t ring = 0, na = 0;
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task task = prm.tasks[prm.pair_ids[it]];
                const int n = task.num_kv_tiles;
                if (n == 0 || sh->abort_flag) continue;
                {   // this CTA's 128 stationary rows of K and V, two 64-column swizzle blocks each
                    wait(BAR_A_EMPTY, (na & 1) ^ 1);
                    const uint32_t afull = lead_bars + 8 * BAR_A_FULL;
                    if (rank == 0) mbar_expect_tx(bars + 8 * BAR_A_FULL, 4 * A_BYTES);
                    const int arow = task.q_begin + BR * (int)rank;
                    tma_load_4d_pair(sA1, &prm.tm_a1, afull, 0, arow, task.h, task.b);
                    tma_load_4d_pair(sA1 + AHALF_BYTES, &prm.tm_a1, afull, 64, arow, task.h, task.b);
                    tma_load_4d_pair(sA2, &prm.tm_a2, afull, 0, arow, task.h, task.b);
                    tma_load_4d_pair(sA2 + AHALF_BYTES, &prm.tm_a2, afull, 64, arow, task.h, task.b);
                    ++na;
                }
                const int64_t ld_base = ((int64_t)task.b * prm.H + task.h) * prm.Nq;   // KEYS: the streamed rows are query rows
                TileCursor cur;
                cur.init(prm.r_begin, prm.r_end, task.range_begin, task.range_count);
                const int np = (n + 1) >> 1;
                for (int p = 0; p < np; ++p) {
                    const Tile t0 = cur.get();
                    cur.next();
                    Tile t1 = t0;                          // odd tail: the second tile is a fully masked copy of the first
                    if (2 * p + 1 < n) { t1 = cur.get(); cur.next(); }
                    {   // {B1, B2} of this CTA's tile, K-major: [B1 h0 | B1 h1 | B2 h0 | B2 h1]
                        const uint32_t slot = ring % NSTAGE;
                        wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                        const uint32_t dst = sRing + slot * SLOT_BYTES, full = lead_bars + 8 * (BAR_KV_FULL + slot);
                        if (rank == 0) mbar_expect_tx(bars + 8 * (BAR_KV_FULL + slot), 2 * SLOT_BYTES + 2 * AUG_STAGE_BYTES);
                        const int row = rank ? t1.key_row : t0.key_row;
                        tma_load_4d_pair(dst, &prm.tm_b1, full, 0, row, task.h, task.b);
                        tma_load_4d_pair(dst + BLK_BYTES, &prm.tm_b1, full, 64, row, task.h, task.b);
                        tma_load_4d_pair(dst + 2 * BLK_BYTES, &prm.tm_b2, full, 0, row, task.h, task.b);
                        tma_load_4d_pair(dst + 3 * BLK_BYTES, &prm.tm_b2, full, 64, row, task.h, task.b);
                        {   // the 16 extra K columns of the tile's rows: -lse/s for X, -delta for Y (slots 0 and 2 hold such tiles)
                            const uint32_t adst = sAug + (slot >> 1) * AUG_STAGE_BYTES;
                            tma_load_2d_pair(adst, &prm.tm_aug1, full, 0, (int)(ld_base + row));
                            tma_load_2d_pair(adst + AUG_TILE_BYTES, &prm.tm_aug2, full, 0, (int)(ld_base + row));
                        }
                        ++ring;
                    }
                    {   // this CTA's column half of the MN-major operands of both tiles
                        const uint32_t slot = ring % NSTAGE;
                        wait(BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                        const uint32_t dst = sRing + slot * SLOT_BYTES, full = lead_bars + 8 * (BAR_KV_FULL + slot);
                        const int col = 64 * (int)rank;
                        {   // [B1(j0) | B2(j0) | B1(j1) | B2(j1)]
                            if (rank == 0) mbar_expect_tx(bars + 8 * (BAR_KV_FULL + slot), 2 * SLOT_BYTES);
                            tma_load_4d_pair(dst, &prm.tm_b1, full, col, t0.key_row, task.h, task.b);
                            tma_load_4d_pair(dst + BLK_BYTES, &prm.tm_b2, full, col, t0.key_row, task.h, task.b);
                            tma_load_4d_pair(dst + 2 * BLK_BYTES, &prm.tm_b1, full, col, t1.key_row, task.h, task.b);
                            tma_load_4d_pair(dst + 3 * BLK_BYTES, &prm.tm_b2, full, col, t1.key_row, task.h, task.b);
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
            const uint32_t a1_lo = ((sA1 >> 4) & 0x3FFF) | LBO_CANON, a2_lo = ((sA2 >> 4) & 0x3FFF) | LBO_CANON;
            const uint32_t ones_lo = ((sOnes >> 4) & 0x3FFF) | LBO_CANON;
            auto aug_lo = [&](uint32_t slot) { return (((sAug + (slot >> 1) * AUG_STAGE_BYTES) >> 4) & 0x3FFF) | LBO_CANON; };
            uint32_t ring = 0, na = 0, c_step = 0;        // ring items consumed; tasks; pair-steps (barrier phases)
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task &tk = prm.tasks[prm.pair_ids[it]];
                const int n = (int)warp_uniform((uint32_t)tk.num_kv_tiles | (sh->abort_flag ? 0x80000000u : 0u));
                if (n <= 0) continue;
                wait(BAR_A_FULL, na & 1);
                ++na;
                tc_fence_after();
                const int np = (n + 1) >> 1;
                uint32_t xslot = 0, b_lo = 0;
                auto issue_x = [&]() {
                    xslot = ring % NSTAGE;
                    wait(BAR_KV_FULL + xslot, (ring / NSTAGE) & 1);
                    tc_fence_after();
                    b_lo = (((sRing + xslot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
                    if (leader) {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {       // [X(j0) | X(j1)] = A1 [B1(j0) ; B1(j1)]^T
                            const uint32_t aoff = ((ks >> 2) * AHALF_BYTES + (ks & 3) * 32) >> 4;
                            const uint32_t boff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                            mma_ss_pair(tmem + TM_X, a1_lo + aoff, DESC_HI, b_lo + boff, DESC_HI, IDESC_XY, ks > 0);
                        }
                        // X -= lse / s of the column's query row (augmentation step)
                            mma_ss_pair(tmem + TM_X, ones_lo, DESC_HI_SW32, aug_lo(xslot), DESC_HI_SW32, IDESC_XY, 1u);
                        tc_commit_pair(bars + 8 * BAR_X_FULL, 3);
                    }
                    __syncwarp();
                    ++ring;
                };
                auto issue_y = [&](bool last) {
                    const uint32_t b2_lo = b_lo + ((2 * BLK_BYTES) >> 4);
                    if (leader) {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {       // [Y(j0) | Y(j1)] = A2 [B2(j0) ; B2(j1)]^T
                            const uint32_t aoff = ((ks >> 2) * AHALF_BYTES + (ks & 3) * 32) >> 4;
                            const uint32_t boff = ((ks >> 2) * BLK_BYTES + (ks & 3) * 32) >> 4;
                            mma_ss_pair(tmem + TM_Y, a2_lo + aoff, DESC_HI, b2_lo + boff, DESC_HI, IDESC_XY, ks > 0);
                        }
                        // Y -= delta of the column's query row
                            mma_ss_pair(tmem + TM_Y, ones_lo, DESC_HI_SW32, aug_lo(xslot) + (AUG_TILE_BYTES >> 4), DESC_HI_SW32, IDESC_XY, 1u);
                        tc_commit_pair(bars + 8 * BAR_Y_FULL, 3);
                        tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + xslot), 3);
                        if (last) tc_commit_pair(bars + 8 * BAR_A_EMPTY, 3);   // every X / Y of this task has been issued
                    }
                    __syncwarp();
                };
                issue_x();
                issue_y(np == 1);
                for (int p = 0; p < np; ++p, ++c_step) {
                    const uint32_t mslot = ring % NSTAGE;
                    wait(BAR_KV_FULL + mslot, (ring / NSTAGE) & 1);
                    ++ring;
                    // MN-major operands, this CTA's 64 columns: streamed row r at r * 128 B, 16-row K steps 2 KB apart
                    const uint32_t m_lo = (((sRing + mslot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_CANON;
                    const uint32_t acc = p > 0 ? 1u : 0u;
                    {
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const uint32_t b2i_lo = m_lo + (((2 * i + 1) * BLK_BYTES) >> 4);
                            const uint32_t tW = tmem + TM_X + i * BC;
                            wait(BAR_W_FULL + i, c_step & 1);
                            tc_fence_after();
                            if (leader) {
#pragma unroll
                                for (int ks = 0; ks < BC / 16; ++ks)    // acc2 += W B2   (dV += P^T dO)
                                    mma_ts_pair(tmem + TM_ACC2, tW + (ks >> 1) * 32 + (ks & 1) * 8, b2i_lo + ks * (2048 >> 4), DESC_HI, IDESC_ACC, acc | (uint32_t)(i > 0) | (ks > 0));
                            }
                            __syncwarp();
                        }
                        if (p + 1 < np) issue_x();                  // overwrites W(p): the pipe executes in order
                    }
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const uint32_t b1i_lo = m_lo + (((2 * i) * BLK_BYTES) >> 4);
                        const uint32_t tZ = tmem + TM_Y + i * BC;
                        wait(BAR_Z_FULL + i, c_step & 1);
                        tc_fence_after();
                        if (leader) {
#pragma unroll
                            for (int ks = 0; ks < BC / 16; ++ks)        // acc1 += Z B1   (dQ += dS K | dK += dS^T Q)
                                mma_ts_pair(tmem + TM_ACC1, tZ + (ks >> 1) * 32 + (ks & 1) * 8, b1i_lo + ks * (2048 >> 4), DESC_HI, IDESC_ACC, acc | (uint32_t)(i > 0) | (ks > 0));
                        }
                        __syncwarp();
                    }
                    if (leader) {
                        tc_commit_pair(bars + 8 * (BAR_KV_EMPTY + mslot), 3);
                        tc_commit_pair(bars + 8 * BAR_ACC_DONE, 3);
                    }
                    __syncwarp();
                    if (p + 1 < np) issue_y(p + 2 == np);           // overwrites Z(p): after the Z MMAs in pipe order
                }
            }
        }
    } else if (warp >= 4) {
        // ================================================= exp / dS / epilogue (both CTAs) ==========================
        const int wg = (warp - 4) >> 2;                            // this warpgroup's tile of every pair-step
        const int row = (threadIdx.x - 128) & (BR - 1);            // stationary row inside this CTA's half = TMEM lane
        const int prow = row + BR * (int)rank;                     // row inside the 256-row tile of the pair
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const float sl2 = prm.scale_log2;
        const uint64_t sl2_2 = pack2(sl2, sl2);
        const uint32_t tX = tmem + lane_base + TM_X + 32 * wg, tY = tmem + lane_base + TM_Y + 32 * wg;   // + 64 i for tile j_i
        uint32_t c_step = 0;
        for (int it = list_begin; it < list_end; ++it) {
            if (sh->abort_flag) break;
            const aj_task task = prm.tasks[prm.pair_ids[it]];
            const int n = task.num_kv_tiles;
            const bool store = prow < task.q_rows;
            const int64_t grow = task.q_begin + prow;
            RowCursor cur;
            cur.init(prm.r_begin, prm.r_end, prm.rows, task.range_begin, task.range_count, prow);
            const int np = (n + 1) >> 1;
            for (int p = 0; p < np; ++p, ++c_step) {
                // streamed rows of the two tiles that this stationary row may see (inside the entry's range and its row interval;
                // PAPER.md:909-914 from the side of the pass)
                int valid[2];
                if (cur.pair_inside()) {
                    valid[0] = valid[1] = cur.pair();
                } else {
                    valid[0] = cur.tile();
                    valid[1] = 2 * p + 1 < n ? cur.tile() : 0;
                }
                // Each warpgroup takes the streamed rows (columns) [32 wg, 32 wg + 32) of BOTH tiles, tile j0 first: W(j0) and
                // Z(j0) are complete after half of the pair-step's exponentials, so the MMAs of tile j0 start while tile j1 is
                // still being computed (with a warpgroup per tile both tiles became ready together, late).  The bf16 W / Z of a
                // warpgroup overwrite the first 16 of the 32 fp32 columns it has just read.
                wait(BAR_X_FULL, c_step & 1);
                tc_fence_after();
                // ---- W = exp2(X s log2e - lse log2e) = p_ab (PAPER.md:842-844 with the forward's L, :945), fp32 in registers
                float w[2][32];
                uint32_t xu2[2][32];
                tmem_ld32(tX, xu2[0]);                         // both tiles in flight: one TMEM round trip per phase
                tmem_ld32(tX + BC, xu2[1]);
                tc_wait_ld(xu2[0], xu2[1]);
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const uint32_t (&xu)[32] = xu2[i];
#pragma unroll
                    for (int c = 0; c < 32; c += 2) {
                        const uint64_t x = fmul2(pack2(xu[c], xu[c + 1]), sl2_2);      // -lse / s of the column is already inside X
                        float x0, x1;                          // (half of these on the FMA pipe was measured slower: DESIGN.md 6d)
                        unpack2(x, x0, x1);
                        w[i][c] = ex2(x0);
                        w[i][c + 1] = ex2(x1);
                    }
                    const int v = valid[i] - 32 * wg;          // of this warpgroup's 32 columns, the first v are seen
                    if (v < 32) {                              // outside the range / the row interval: p = 0 (selected after the
#pragma unroll                                                 // exponential: the masked operands may be anything, even inf - inf)
                        for (int c = 0; c < 32; ++c) if (c >= v) w[i][c] = 0.f;
                    }
                    {                                          // bf16 W = P^T, the A operand of dV += P^T dO
                        uint32_t wk[16];
#pragma unroll
                        for (int c = 0; c < 16; ++c) wk[c] = pack_bf16(w[i][2 * c], w[i][2 * c + 1]);
                        tmem_st16(tX + BC * i, wk);
                        tc_wait_st();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(lead_bars + 8 * (BAR_W_FULL + i));
                    }
                }
                // ---- Z = W o (Y - delta) = dS / s
                wait(BAR_Y_FULL, c_step & 1);
                tc_fence_after();
                uint32_t yu2[2][32];
                tmem_ld32(tY, yu2[0]);
                tmem_ld32(tY + BC, yu2[1]);
                tc_wait_ld(yu2[0], yu2[1]);
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const uint32_t (&yu)[32] = yu2[i];
                    uint32_t zk[16];
#pragma unroll
                    for (int c = 0; c < 32; c += 2) {
                        const uint64_t y = pack2(yu[c], yu[c + 1]);                 // -delta is inside Y
                        const uint64_t z = fmul2(pack2(w[i][c], w[i][c + 1]), y);
                        float z0, z1;
                        unpack2(z, z0, z1);
                        zk[c >> 1] = pack_bf16(z0, z1);
                    }
                    const int v = valid[i] - 32 * wg;
                    if (v < 32) {                              // masked columns: Z = 0 whatever Y held (a branch, not 32 selects)
#pragma unroll
                        for (int k = 0; k < 16; ++k) zk[k] = 2 * k >= v ? 0u : (2 * k + 1 >= v ? (zk[k] & 0xffffu) : zk[k]);
                    }
                    tmem_st16(tY + BC * i, zk);
                    tc_wait_st();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(lead_bars + 8 * (BAR_Z_FULL + i));
                }
            }
            // ---- epilogue: acc1 * s -> dQ | dK, acc2 -> dV; each warpgroup writes one 64-column half ----
            __nv_bfloat16 *o1 = (__nv_bfloat16 *)prm.out1.ptr + task.b * prm.out1.stride_b + task.h * prm.out1.stride_h + grow * prm.out1.stride_n;
            __nv_bfloat16 *o2 = (__nv_bfloat16 *)prm.out2.ptr + task.b * prm.out2.stride_b + task.h * prm.out2.stride_h + grow * prm.out2.stride_n;
            if (n == 0) {                                           // a row without keys / a key no row sees: zeros
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = 8 * wg; c < 8 * wg + 8; ++c) { ((uint4 *)o1)[c] = z; ((uint4 *)o2)[c] = z; }
                }
                continue;
            }
            // A parity wait is sound only if the barrier is known to be at most one phase away: this thread consumed Y of the
            // last pair-step, which the in-order pipe produced after committing ACC_DONE of the pair-step before, and the next
            // phase needs this thread's next hand-over.
            wait(BAR_ACC_DONE, (c_step - 1) & 1);
            tc_fence_after();
#pragma unroll 1
            for (int cb = 64 * wg; cb < 64 * wg + 64; cb += 32) {
                uint32_t a1[32], a2[32];
                tmem_ld32(tmem + lane_base + TM_ACC1 + cb, a1);
                tmem_ld32(tmem + lane_base + TM_ACC2 + cb, a2);
                tc_wait_ld(a1, a2);
                if (store) {
#pragma unroll
                    for (int v4 = 0; v4 < 4; ++v4) {
                        uint32_t w1[4], w2[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int c = v4 * 8 + 2 * e;
                            w1[e] = pack_bf16(__uint_as_float(a1[c]) * prm.scale, __uint_as_float(a1[c + 1]) * prm.scale);
                            w2[e] = pack_bf16(__uint_as_float(a2[c]), __uint_as_float(a2[c + 1]));
                        }
                        *(uint4 *)(o1 + cb + v4 * 8) = make_uint4(w1[0], w1[1], w1[2], w1[3]);
                        *(uint4 *)(o2 + cb + v4 * 8) = make_uint4(w2[0], w2[1], w2[2], w2[3]);
                    }
                }
            }
            tc_fence_before();
            named_bar_sync(3, 256);          // the accumulators and the A columns are free only when both warpgroups are done
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


// ======================================================================================================================
// dQ pass, second form ("tile ping-pong"): the same computation as attn_bwd_umma_pair_kernel<false>, with the streamed tiles
// taken ONE AT A TIME and the two exp / dS warpgroups on ALTERNATE tiles.  The A operands of X and Y sit in TMEM, so their
// MMAs do not need N = 128 to stay off the shared-memory port; with N = 64 (cta_group::2: each CTA stages 32 rows of the
// tile's K and V) X(j) | Y(j) of tile j occupy one 64 + 64 column buffer and the two buffers alternate:
//     issue order   X(j+1), Y(j+1) [buffer (j+1) & 1]   then   acc1 += Z(j) K(j) [buffer j & 1]
// A warpgroup has two tile periods (2 x 768 clk of tensor work) to turn X, Y of its tile into Z, and nothing on the tensor
// pipe waits for it except its own tile's last MMA.  In the pair-step form the chain Y(p) -> Z(p) -> Z(p) K -> Y(p+1) is
// serial (X and Y are single-buffered at 128 + 128 columns) and the pipe idles a third of the time (ncu: 65 %).
// TMEM: acc1 128 | bf16 Q 64 + dO 64 | X(b0) X(b1) 128 | Y(b0) Y(b1) 128.  Ring: 8 slots of 24 KB per tile and CTA:
// [K rows 32c..32c+32: h0 | h1 | V rows likewise: h0 | h1 (4 KB each, K-major) | K(j) columns 64c..64c+64 (8 KB, MN-major)].
constexpr int DQ_NSTAGE = 8;
constexpr uint32_t DQ_HBLK = 32 * 64 * 2;              // 4 KB: 32 streamed rows x 64 columns
constexpr uint32_t DQ_SLOT = 4 * DQ_HBLK + BLK_BYTES;  // 24 KB
constexpr uint32_t DQ_SMEM_TILES = DQ_NSTAGE * DQ_SLOT;
constexpr uint32_t DQ_SMEM_TOTAL = DQ_SMEM_TILES + 1024 + 512;
constexpr uint32_t IDESC_XY64 = make_idesc(BC, false);     // 256 x 64 x 16, B K-major (32 streamed rows per CTA)
enum {
    DQ_A_FULL = 0,                              // leader: 16 warps stored their Q / dO rows to TMEM
    DQ_KV_FULL,                                 // leader, x DQ_NSTAGE
    DQ_KV_EMPTY = DQ_KV_FULL + DQ_NSTAGE,       // both
    DQ_XY_FULL = DQ_KV_EMPTY + DQ_NSTAGE,       // both, x2 (buffer)
    DQ_Z_FULL = DQ_XY_FULL + 2,                 // leader, x2: Z stored by the tile's warpgroup in both CTAs
    DQ_ACC_DONE = DQ_Z_FULL + 2,                // both, x2 (buffer): every MMA up to and including the tile's Z K is complete
    DQ_NUM_BARS = DQ_ACC_DONE + 2
};
static_assert(DQ_NUM_BARS <= NUM_BARS + 16, "barrier array");
struct DqShared {
    uint64_t bars[DQ_NUM_BARS];
    uint32_t tmem_base;
    int abort_flag;
};
static_assert(sizeof(DqShared) <= 512, "struct DqShared outgrew its reservation");

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
attn_bwd_dq_pair_kernel(const __grid_constant__ BwdPairParams prm) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;
    DqShared *sh = reinterpret_cast<DqShared *>(smem_raw + (tiles - raw) + DQ_SMEM_TILES);
    const uint32_t sRing = tiles;
    const uint32_t bars = smem_u32(sh->bars);
    const PairWaiter wait{bars, &sh->abort_flag, prm.err, 250};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const uint32_t lead_bars = mapa(bars, 0);
    const int pair = blockIdx.x >> 1;
    const int list_begin = prm.pair_off[pair], list_end = prm.pair_off[pair + 1];

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * DQ_A_FULL, 16);
        for (int i = 0; i < DQ_NSTAGE; ++i) { mbar_init(bars + 8 * (DQ_KV_FULL + i), 1); mbar_init(bars + 8 * (DQ_KV_EMPTY + i), 1); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bars + 8 * (DQ_XY_FULL + b), 1);
            mbar_init(bars + 8 * (DQ_Z_FULL + b), 8);
            mbar_init(bars + 8 * (DQ_ACC_DONE + b), 1);
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

    if (warp == 0) {
        // ================================================= TMA producer (both CTAs) ================================
        if (lane == 0) {
            prefetch_tmap(&prm.tm_b1); prefetch_tmap(&prm.tm_b2); prefetch_tmap(&prm.tm_b1h); prefetch_tmap(&prm.tm_b2h);
            uint32_t ring = 0;
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task task = prm.tasks[prm.pair_ids[it]];
                const int n = task.num_kv_tiles;
                if (n == 0 || sh->abort_flag) continue;
                TileCursor cur;
                cur.init(prm.r_begin, prm.r_end, task.range_begin, task.range_count);
                for (int j = 0; j < n; ++j, cur.next(), ++ring) {
                    const Tile t = cur.get();
                    const uint32_t slot = ring % DQ_NSTAGE;
                    wait(DQ_KV_EMPTY + slot, ((ring / DQ_NSTAGE) & 1) ^ 1);
                    const uint32_t dst = sRing + slot * DQ_SLOT, full = lead_bars + 8 * (DQ_KV_FULL + slot);
                    if (rank == 0) mbar_expect_tx(bars + 8 * (DQ_KV_FULL + slot), 2 * DQ_SLOT);
                    const int row = t.key_row + 32 * (int)rank;     // this CTA's 32 of the tile's 64 keys (B operand split by N)
                    tma_load_4d_pair(dst, &prm.tm_b1h, full, 0, row, task.h, task.b);
                    tma_load_4d_pair(dst + DQ_HBLK, &prm.tm_b1h, full, 64, row, task.h, task.b);
                    tma_load_4d_pair(dst + 2 * DQ_HBLK, &prm.tm_b2h, full, 0, row, task.h, task.b);
                    tma_load_4d_pair(dst + 3 * DQ_HBLK, &prm.tm_b2h, full, 64, row, task.h, task.b);
                    tma_load_4d_pair(dst + 4 * DQ_HBLK, &prm.tm_b1, full, 64 * (int)rank, t.key_row, task.h, task.b);
                }
            }
        }
    } else if (warp == 1) {
        // ================================================= MMA issuer (leader CTA) ==================================
        if (rank == 0) {
            const bool leader = elect_one();
            uint32_t ring = 0, na = 0;                    // ring = tiles before this task = global tile index base
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task &tk = prm.tasks[prm.pair_ids[it]];
                const int n = (int)warp_uniform((uint32_t)tk.num_kv_tiles | (sh->abort_flag ? 0x80000000u : 0u));
                if (n <= 0) continue;
                wait(DQ_A_FULL, na & 1);
                ++na;
                tc_fence_after();
                auto issue_xy = [&](uint32_t g) {         // X(g) = Q K(g)^T, Y(g) = dO V(g)^T into buffer g & 1
                    const uint32_t slot = g % DQ_NSTAGE, b = g & 1;
                    wait(DQ_KV_FULL + slot, (g / DQ_NSTAGE) & 1);
                    tc_fence_after();
                    const uint32_t k_lo = (((sRing + slot * DQ_SLOT) >> 4) & 0x3FFF) | LBO_CANON, v_lo = k_lo + ((2 * DQ_HBLK) >> 4);
                    if (leader) {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            const uint32_t boff = ((ks >> 2) * DQ_HBLK + (ks & 3) * 32) >> 4;
                            mma_ts_pair(tmem + TM_X + BC * b, tmem + TM_A1 + ks * 8, k_lo + boff, DESC_HI, IDESC_XY64, ks > 0);
                        }
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            const uint32_t boff = ((ks >> 2) * DQ_HBLK + (ks & 3) * 32) >> 4;
                            mma_ts_pair(tmem + TM_Y + BC * b, tmem + TM_A2 + ks * 8, v_lo + boff, DESC_HI, IDESC_XY64, ks > 0);
                        }
                        tc_commit_pair(bars + 8 * (DQ_XY_FULL + b), 3);
                    }
                    __syncwarp();
                };
                issue_xy(ring);
                for (int j = 0; j < n; ++j) {
                    const uint32_t g = ring + (uint32_t)j, slot = g % DQ_NSTAGE, b = g & 1;
                    if (j + 1 < n) issue_xy(g + 1);
                    const uint32_t m_lo = (((sRing + slot * DQ_SLOT + 4 * DQ_HBLK) >> 4) & 0x3FFF) | LBO_CANON;
                    wait(DQ_Z_FULL + b, (g >> 1) & 1);
                    tc_fence_after();
                    if (leader) {
#pragma unroll
                        for (int ks = 0; ks < BC / 16; ++ks)        // acc1 += Z K   (dQ += dS K)
                            mma_ts_pair(tmem + TM_ACC1, tmem + TM_Y + BC * b + ks * 8, m_lo + ks * (2048 >> 4), DESC_HI, IDESC_ACC, (uint32_t)(j > 0) | (ks > 0));
                        tc_commit_pair(bars + 8 * (DQ_KV_EMPTY + slot), 3);
                        tc_commit_pair(bars + 8 * (DQ_ACC_DONE + b), 3);
                    }
                    __syncwarp();
                }
                ring += (uint32_t)n;
            }
        }
    } else if (warp >= 4) {
        // ================================================= exp / dS / epilogue (both CTAs) ==========================
        const int wg = (warp - 4) >> 2;                            // takes the tiles whose global index has this parity
        const int row = (threadIdx.x - 128) & (BR - 1);
        const int prow = row + BR * (int)rank;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const float sl2 = prm.scale_log2;
        const uint64_t sl2_2 = pack2(sl2, sl2);
        const uint32_t z_full = lead_bars + 8 * (DQ_Z_FULL + wg);
        const uint32_t tX = tmem + lane_base + TM_X + BC * wg, tY = tmem + lane_base + TM_Y + BC * wg;
        uint32_t g0 = 0;                                           // tiles before this task
        for (int it = list_begin; it < list_end; ++it) {
            if (sh->abort_flag) break;
            const aj_task task = prm.tasks[prm.pair_ids[it]];
            const int n = task.num_kv_tiles;
            const bool store = prow < task.q_rows;
            const int64_t grow = task.q_begin + prow;
            uint64_t myl_2 = 0ull, myd_2 = 0ull;
            if (n > 0) {
                float2 my = make_float2(0.f, 0.f);
                if (store) my = prm.ld[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow];
                myl_2 = pack2(-my.x, -my.x); myd_2 = pack2(-my.y, -my.y);
                // this thread's row of Q (warpgroup 0) or dO (warpgroup 1) as a bf16 A operand in TMEM
                const aj_tensor &src = wg ? prm.a2 : prm.a1;
                const uint4 *rowp = (const uint4 *)((const __nv_bfloat16 *)src.ptr + task.b * src.stride_b + task.h * src.stride_h + grow * src.stride_n);
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    uint32_t ra[32];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const uint4 u = store ? rowp[half * 8 + i] : make_uint4(0, 0, 0, 0);
                        ra[4 * i] = u.x; ra[4 * i + 1] = u.y; ra[4 * i + 2] = u.z; ra[4 * i + 3] = u.w;
                    }
                    tmem_st32(tmem + lane_base + (wg ? TM_A2 : TM_A1) + 32 * half, ra);
                }
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(lead_bars + 8 * DQ_A_FULL);
            }
            RowCursor cur;
            cur.init(prm.r_begin, prm.r_end, prm.rows, task.range_begin, task.range_count, prow);
            for (int j = 0; j < n; ++j) {
                const uint32_t g = g0 + (uint32_t)j;
                const int valid = cur.tile();                      // keys of the tile this row may see
                if ((int)(g & 1) != wg) continue;                  // the other warpgroup's tile
                wait(DQ_XY_FULL + wg, (g >> 1) & 1);
                tc_fence_after();
                uint32_t zk[32];
                uint32_t xh[2][32], yh[2][32];
                tmem_ld32(tX, xh[0]);
                tmem_ld32(tY, yh[0]);
                tc_wait_ld(xh[0], yh[0]);
                tmem_ld32(tX + 32, xh[1]);                       // the second half is in flight under the first half's arithmetic
                tmem_ld32(tY + 32, yh[1]);
#pragma unroll
                for (int hb = 0; hb < 2; ++hb) {
                    if (hb == 1) tc_wait_ld(xh[1], yh[1]);
                    const uint32_t (&xu)[32] = xh[hb];
                    const uint32_t (&yu)[32] = yh[hb];
#pragma unroll
                    for (int c = 0; c < 32; c += 2) {
                        // W = exp2(S s log2e - lse log2e) = p_ab;  Z = W (dP - delta) = dS / s
                        const uint64_t x = ffma2(pack2(xu[c], xu[c + 1]), sl2_2, myl_2);
                        float x0, x1;
                        unpack2(x, x0, x1);
                        const uint64_t z = fmul2(pack2(ex2(x0), ex2(x1)), fadd2(pack2(yu[c], yu[c + 1]), myd_2));
                        float z0, z1;
                        unpack2(z, z0, z1);
                        zk[(32 * hb + c) >> 1] = pack_bf16(z0, z1);
                    }
                }
                if (valid < BC) {                              // masked columns: Z = 0, selected after the exponential (a branch, not 64 selects)
#pragma unroll
                    for (int k = 0; k < 32; ++k) zk[k] = 2 * k >= valid ? 0u : (2 * k + 1 >= valid ? (zk[k] & 0xffffu) : zk[k]);
                }
                tmem_st32(tY, zk);
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(z_full);
            }
            // ---- epilogue: acc1 * s -> dQ; each warpgroup writes one 64-column half ----
            __nv_bfloat16 *o1 = (__nv_bfloat16 *)prm.out1.ptr + task.b * prm.out1.stride_b + task.h * prm.out1.stride_h + grow * prm.out1.stride_n;
            if (n == 0) {
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = 8 * wg; c < 8 * wg + 8; ++c) ((uint4 *)o1)[c] = z;
                }
                continue;
            }
            // The warpgroup of the last tile saw X, Y of that tile, which the in-order pipe produced after the Z K of the tile
            // three before (the previous phase of this buffer's barrier is the tile two before): after the named barrier both
            // warpgroups know that the barrier is at most one phase away.
            named_bar_sync(3, 256);
            {
                const uint32_t gl = g0 + (uint32_t)n - 1;
                wait(DQ_ACC_DONE + (gl & 1), (gl >> 1) & 1);
                tc_fence_after();
            }
            g0 += (uint32_t)n;
#pragma unroll 1
            for (int cb = 64 * wg; cb < 64 * wg + 64; cb += 32) {
                uint32_t a1[32];
                tmem_ld32(tmem + lane_base + TM_ACC1 + cb, a1);
                tc_wait_ld(a1);
                if (store) {
#pragma unroll
                    for (int v4 = 0; v4 < 4; ++v4) {
                        uint32_t w1[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int c = v4 * 8 + 2 * e;
                            w1[e] = pack_bf16(__uint_as_float(a1[c]) * prm.scale, __uint_as_float(a1[c + 1]) * prm.scale);
                        }
                        *(uint4 *)(o1 + cb + v4 * 8) = make_uint4(w1[0], w1[1], w1[2], w1[3]);
                    }
                }
            }
            tc_fence_before();
            named_bar_sync(4, 256);          // the accumulator and the A columns are free only when both warpgroups are done
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

cudaError_t launch_bwd_umma_pair(const BwdPairParams &prm, bool keys, int num_pairs, cudaStream_t stream) {
    if (num_pairs <= 0 || prm.num_tasks <= 0) return cudaSuccess;
    static std::atomic<uint64_t> configured[2];
    if (keys) {
        if (cudaError_t e = ensure_dynamic_smem(attn_bwd_umma_pair_kernel<true>, (int)Cfg<true>::SMEM_TOTAL, configured[1])) return e;
        attn_bwd_umma_pair_kernel<true><<<2 * num_pairs, NTHREADS, Cfg<true>::SMEM_TOTAL, stream>>>(prm);
    } else {                            // (the pair-step form of this pass, attn_bwd_umma_pair_kernel<false>, was measured slower: DESIGN.md 6d)
        static std::atomic<uint64_t> configured_dq{0};
        if (cudaError_t e = ensure_dynamic_smem(attn_bwd_dq_pair_kernel, (int)DQ_SMEM_TOTAL, configured_dq)) return e;
        attn_bwd_dq_pair_kernel<<<2 * num_pairs, NTHREADS, DQ_SMEM_TOTAL, stream>>>(prm);
    }
    return cudaGetLastError();
}

}  // namespace aj
