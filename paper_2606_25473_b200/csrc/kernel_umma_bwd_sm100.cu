// bf16 primal backward of masked attention for sm_100a: TMA -> shared-memory ring -> tcgen05.mma with
// TMEM accumulators.  Same formulas as kernel_simt_bwd.cu (the VJP of Eq. 42):
//     p_ab = exp(s <q_a, k_b> - lse_a),  dP_ab = <dO_a, v_b>,  dS_ab = p_ab (dP_ab - delta_a),  delta_a = <dO_a, O_a>
//     dQ_a = s sum_b dS_ab k_b ;   dK_b = s sum_a dS_ab q_a ;   dV_b = sum_a p_ab dO_a
// Two passes of ONE kernel, because the two are the same computation with the roles swapped:
//   a CTA keeps 128 STATIONARY rows (A1, A2; in shared memory, or in TMEM in the dQ pass) and streams 64-row tiles (B1, B2)
//   of the other side:
//     X  = A1 B1^T,  Y = A2 B2^T            2 x 8 MMAs (M128 N64 K16), B from shared memory          -> TMEM
//     W  = exp2(X s log2e - lse log2e),  Z = W o (Y - delta)         softmax warps, thread = stationary row = TMEM lane
//     acc1 += Z B1   (and acc2 += W B2)     4 (+4) MMAs (M128 N128 K16), A = bf16 Z / W in TMEM, B MN-major
//   KEYS = false: stationary = query rows (A1 = Q, A2 = dO), streamed = keys (B1 = K, B2 = V): acc1 = dQ / s; lse and
//                 delta belong to the thread's own row.
//   KEYS = true:  stationary = keys (A1 = K, A2 = V), streamed = query rows (B1 = Q, B2 = dO): X = S^T, Y = dP^T,
//                 acc1 = dK / s, acc2 = dV; lse and delta belong to the COLUMNS and are staged in shared memory per tile.
//                 The tasks come from the transposed schedule (key tiles with the row ranges that see them).
// S and dP are therefore computed twice (7 contractions instead of the minimal 5) in exchange for no atomics and no
// cross-CTA reduction of dQ.  X/Y are double-buffered in TMEM (acc1 128 | acc2 128 | X0 Y0 X1 Y1 64 columns each), so
// the MMAs of tile j + 1 run under the exp / dS work of tile j.  Roles (12 warps): warp 0 TMA producer, warp 1 MMA issuer,
// warp 2 TMEM allocator, warps 4-7 and 8-11 two exp / dS / epilogue warpgroups that each take 32 of a tile's 64 streamed
// rows (the columns are independent: there is no running max).  Tasks are assigned to the CTAs by the host, head by head
// and most expensive first (assign_workers), so that all CTAs stream the same head's operands through L2 at the same time.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

#include "kernels.hpp"
#include "umma_ptx.cuh"

namespace aj {

namespace {

using namespace ptx;

constexpr int BR = UMMA_TILE_Q;        // 128 stationary rows
constexpr int BC = UMMA_TILE_K;        // 64 streamed rows per tile
constexpr int NSTAGE_MAX = 8;
constexpr uint32_t AHALF_BYTES = BR * 64 * 2;      // one 64-column swizzle block of a stationary operand: 16 KB
constexpr uint32_t BHALF_BYTES = BC * 64 * 2;      // 8 KB
// Head dimension D = 128 (two 64-column swizzle blocks per operand row) or 64 (one block; the accumulators use the first 64
// of their 128 TMEM columns).
template <int D> struct Cfg {
    static_assert(D == 64 || D == 128, "d must be 64 or 128");
    static constexpr int NB = D / 64;                                    // swizzle blocks per operand row
    static constexpr int NSTAGE = D == 128 ? 4 : 8;   // ring slots [B1 h0 | B1 h1 | B2 h0 | B2 h1] of 32 KB | [B1 | B2] of 16 KB (6 slots of
                                                      // 32 KB in the dQ pass, whose stationary operands live in TMEM, measured no faster:
                                                      // 13.05 M against 12.69 M cycles)
    static constexpr uint32_t A_BYTES = BR * D * 2;                      // 32 KB | 16 KB
    static constexpr uint32_t SLOT_BYTES = 2 * NB * BHALF_BYTES;         // 32 KB | 16 KB
    static constexpr uint32_t SMEM_TILES = 2 * A_BYTES + NSTAGE * SLOT_BYTES;   // 192 KB | 160 KB
    static constexpr uint32_t SMEM_TOTAL = SMEM_TILES + 1024 /*align*/ + 2048 /*struct Shared*/;
};
constexpr int NTHREADS = 384;               // warps 0-3: TMA / MMA / TMEM alloc / idle; warps 4-7 and 8-11: exp / dS warpgroups 0, 1

constexpr uint32_t TM_ACC1 = 0, TM_ACC2 = 128, TM_X0 = 256, TM_Y0 = 320, TM_BUF = 128;   // X1 = X0 + 128, Y1 = Y0 + 128
// dQ pass: there is no acc2, and its 128 columns hold the stationary operands themselves as bf16 A operands (64 columns
// each): the X / Y MMAs then read A from TMEM, which takes their 4 KB per instruction off the shared-memory port (the
// port, not the tensor pipe, bounds the N = 64 shared-memory-operand form: 6 KB per 32 clk of math at 128 B/clk).
constexpr uint32_t TM_A1 = 128, TM_A2 = 192;

enum {
    BAR_A_FULL = 0, BAR_A_EMPTY,
    BAR_B_FULL, BAR_B_EMPTY = BAR_B_FULL + NSTAGE_MAX,
    BAR_X_FULL = BAR_B_EMPTY + NSTAGE_MAX,      // x2: X, Y of the buffer complete
    BAR_W_FULL = BAR_X_FULL + 2,            // x2: Z (and W) stored by the four softmax warps
    BAR_ACC_DONE = BAR_W_FULL + 2,          // x2 (by TMEM buffer): every MMA up to and including the tile's is complete
    NUM_BARS = BAR_ACC_DONE + 2
};

__host__ __device__ constexpr uint32_t make_idesc(int n, bool b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(BR >> 4) << 24);
}
constexpr uint32_t IDESC_XY = make_idesc(BC, false);     // 128 x  64 x 16, A and B K-major
// acc += Z B1 / W B2 is 128 x D x 16, A from TMEM, B MN-major: make_idesc(D, true)
constexpr uint32_t DESC_HI = desc_hi(1024);
constexpr uint32_t LBO_K = desc_lo_lbo(16);              // K-major with 128 B swizzle: unused, canonical value
constexpr uint32_t LBO_MN = desc_lo_lbo(BHALF_BYTES);    // MN-major: the two 64-column blocks of a streamed operand are 8 KB apart

struct Shared {
    uint64_t bars[NUM_BARS];
    uint32_t tmem_base;
    int abort_flag;
    alignas(16) float stage[2][2][BC];     // KEYS pass: [buffer][0 = lse * log2e (+inf past the range end), 1 = delta][streamed row]
};
static_assert(sizeof(Shared) <= 2048, "struct Shared outgrew its reservation");

// Walks the streamed tiles of a task: its ranges [rb, rb + rc), each cut into BC-row tiles from its start.
struct TileCursor {
    const int32_t *b, *e;
    int r, rend, m, mend;
    __device__ void init(const int32_t *begin, const int32_t *end, int rb, int rc) {
        b = begin; e = end; r = rb; rend = rb + rc;
        if (r < rend) { m = b[r]; mend = e[r]; } else { m = 0; mend = 0; }
    }
    __device__ int row() const { return m; }
    __device__ int valid() const { return min(BC, mend - m); }
    __device__ void next() {
        m += BC;
        if (m >= mend) { ++r; if (r < rend) { m = b[r]; mend = e[r]; } }
    }
};

template <bool KEYS, int D>
__global__ void __launch_bounds__(NTHREADS, 1)
attn_bwd_umma_kernel(const __grid_constant__ BwdUmmaParams prm) {
    using C = Cfg<D>;
    constexpr int NB = C::NB;
    constexpr uint32_t A_BYTES = C::A_BYTES, SLOT_BYTES = C::SLOT_BYTES, SMEM_TILES = C::SMEM_TILES;
    constexpr uint32_t IDESC_ACC = make_idesc(D, true);
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;
    Shared *sh = reinterpret_cast<Shared *>(smem_raw + (tiles - raw) + SMEM_TILES);
    constexpr int NSTAGE = C::NSTAGE;
    const uint32_t sA1 = tiles, sA2 = tiles + A_BYTES, sRing = tiles + 2 * A_BYTES;
    const uint32_t bars = smem_u32(sh->bars);
    const Waiter wait{bars, &sh->abort_flag, prm.err};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int list_begin = prm.cta_off[blockIdx.x], list_end = prm.cta_off[blockIdx.x + 1];

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * BAR_A_FULL, KEYS ? 1 : 8);     // TMA transaction | one arrive per exp / dS warp (rows stored to TMEM)
        mbar_init(bars + 8 * BAR_A_EMPTY, 1);
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bars + 8 * (BAR_B_FULL + i), 1); mbar_init(bars + 8 * (BAR_B_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(bars + 8 * (BAR_X_FULL + i), 1); mbar_init(bars + 8 * (BAR_W_FULL + i), 8); }
        mbar_init(bars + 8 * BAR_ACC_DONE, 1);
        mbar_init(bars + 8 * (BAR_ACC_DONE + 1), 1);
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
            prefetch_tmap(&prm.tm_a1); prefetch_tmap(&prm.tm_a2); prefetch_tmap(&prm.tm_b1); prefetch_tmap(&prm.tm_b2);
            uint32_t ring = 0, na = 0;
            for (int it = list_begin; it < list_end; ++it) {
                const aj_task task = prm.tasks[prm.cta_ids[it]];
                const int n = task.num_kv_tiles;
                if (n == 0 || sh->abort_flag) continue;
                if (KEYS) {
                    wait(BAR_A_EMPTY, (na & 1) ^ 1);
                    const uint32_t afull = bars + 8 * BAR_A_FULL;
                    mbar_expect_tx(afull, 2 * A_BYTES);
                    tma_load_4d(sA1, &prm.tm_a1, afull, 0, task.q_begin, task.h, task.b);
                    if (NB == 2) tma_load_4d(sA1 + AHALF_BYTES, &prm.tm_a1, afull, 64, task.q_begin, task.h, task.b);
                    tma_load_4d(sA2, &prm.tm_a2, afull, 0, task.q_begin, task.h, task.b);
                    if (NB == 2) tma_load_4d(sA2 + AHALF_BYTES, &prm.tm_a2, afull, 64, task.q_begin, task.h, task.b);
                    ++na;
                }
                TileCursor cur;
                cur.init(prm.r_begin, prm.r_end, task.range_begin, task.range_count);
                for (int j = 0; j < n; ++j, cur.next(), ++ring) {
                    const uint32_t slot = ring % NSTAGE;
                    wait(BAR_B_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1);
                    const uint32_t dst = sRing + slot * SLOT_BYTES, full = bars + 8 * (BAR_B_FULL + slot);
                    mbar_expect_tx(full, SLOT_BYTES);
                    const int row = cur.row();
                    tma_load_4d(dst, &prm.tm_b1, full, 0, row, task.h, task.b);
                    if (NB == 2) tma_load_4d(dst + BHALF_BYTES, &prm.tm_b1, full, 64, row, task.h, task.b);
                    tma_load_4d(dst + NB * BHALF_BYTES, &prm.tm_b2, full, 0, row, task.h, task.b);
                    if (NB == 2) tma_load_4d(dst + 3 * BHALF_BYTES, &prm.tm_b2, full, 64, row, task.h, task.b);
                }
            }
        }
    } else if (warp == 1) {
        // ================================================= MMA issuer ============================================
        // Every lane runs the control flow (counters and descriptors stay warp-uniform), one elected lane issues.
        const bool leader = elect_one();
        const uint32_t a1_lo = ((sA1 >> 4) & 0x3FFF) | LBO_K, a2_lo = ((sA2 >> 4) & 0x3FFF) | LBO_K;
        uint32_t ring = 0, na = 0, g = 0;   // g = tiles issued so far (selects the X/Y buffer and the barrier phases)
        auto issue_xy = [&](uint32_t gj, uint32_t item) {
            const uint32_t slot = item % NSTAGE;
            wait(BAR_B_FULL + slot, (item / NSTAGE) & 1);
            tc_fence_after();
            const uint32_t b1_lo = (((sRing + slot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_K, b2_lo = b1_lo + ((NB * BHALF_BYTES) >> 4);
            const uint32_t tX = tmem + TM_X0 + (gj & 1) * TM_BUF, tY = tmem + TM_Y0 + (gj & 1) * TM_BUF;
            if (leader) {
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t aoff = ((ks >> 2) * AHALF_BYTES + (ks & 3) * 32) >> 4;
                    const uint32_t boff = ((ks >> 2) * BHALF_BYTES + (ks & 3) * 32) >> 4;
                    if (KEYS) {
                        mma_ss(tX, a1_lo + aoff, DESC_HI, b1_lo + boff, DESC_HI, IDESC_XY, ks > 0);   // X = A1 B1^T  (S^T)
                        mma_ss(tY, a2_lo + aoff, DESC_HI, b2_lo + boff, DESC_HI, IDESC_XY, ks > 0);   // Y = A2 B2^T  (dP^T)
                    } else {
                        mma_ts(tX, tmem + TM_A1 + ks * 8, b1_lo + boff, DESC_HI, IDESC_XY, ks > 0);   // S  = Q K^T, Q from TMEM
                        mma_ts(tY, tmem + TM_A2 + ks * 8, b2_lo + boff, DESC_HI, IDESC_XY, ks > 0);   // dP = dO V^T
                    }
                }
                tc_commit(bars + 8 * (BAR_X_FULL + (gj & 1)));
            }
            __syncwarp();
        };
        for (int it = list_begin; it < list_end; ++it) {
            const int n = (int)warp_uniform((uint32_t)prm.tasks[prm.cta_ids[it]].num_kv_tiles | (sh->abort_flag ? 0x80000000u : 0u));
            if (n <= 0) continue;
            wait(BAR_A_FULL, na & 1);
            ++na;
            tc_fence_after();
            issue_xy(g, ring);
            for (int j = 0; j < n; ++j) {
                const uint32_t gj = g + j, b = gj & 1, item = ring + j, slot = item % NSTAGE;
                if (j + 1 < n) issue_xy(gj + 1, item + 1);
                else if (leader) tc_commit(bars + 8 * BAR_A_EMPTY);      // every X, Y of this task has been issued
                // streamed tile as MN-major B operand: row r at r*128 bytes inside each 64-column block, 16-row K steps 2 KB apart
                const uint32_t b1_lo = (((sRing + slot * SLOT_BYTES) >> 4) & 0x3FFF) | LBO_MN, b2_lo = b1_lo + ((NB * BHALF_BYTES) >> 4);
                const uint32_t tW = tmem + TM_X0 + b * TM_BUF, tZ = tmem + TM_Y0 + b * TM_BUF;
                const uint32_t acc = j > 0 ? 1u : 0u;
                wait(BAR_W_FULL + b, (gj >> 1) & 1);
                tc_fence_after();
                if (leader) {
#pragma unroll
                    // bf16 Z / W of streamed rows [32 h, 32 h + 32) sit in columns [32 h, 32 h + 16) of the Y / X buffer
                    // (each exp / dS warpgroup writes inside the fp32 columns it has read)
                    for (int ks = 0; ks < BC / 16; ++ks)        // acc1 += Z B1   (dQ += dS K | dK += dS^T Q)
                        mma_ts(tmem + TM_ACC1, tZ + (ks >> 1) * 32 + (ks & 1) * 8, b1_lo + ks * (2048 >> 4), DESC_HI, IDESC_ACC, acc | (ks > 0));
                    if (KEYS) {
#pragma unroll
                        for (int ks = 0; ks < BC / 16; ++ks)    // acc2 += W B2   (dV += P^T dO)
                            mma_ts(tmem + TM_ACC2, tW + (ks >> 1) * 32 + (ks & 1) * 8, b2_lo + ks * (2048 >> 4), DESC_HI, IDESC_ACC, acc | (ks > 0));
                    }
                    tc_commit(bars + 8 * (BAR_B_EMPTY + slot));
                    tc_commit(bars + 8 * (BAR_ACC_DONE + b));
                }
                __syncwarp();
            }
            g += n;
            ring += n;
        }
    } else if (warp >= 4) {
        // ================================================= exp / dS / epilogue (thread = stationary row = TMEM lane) ==
        const int wg = (warp - 4) >> 2;                            // takes the tiles whose TMEM buffer is wg
        const int row = (threadIdx.x - 128) & (BR - 1);
        const int st = row;                                        // staging duty in the KEYS pass: 0..63 lse, 64..127 delta
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const float sl2 = prm.scale_log2;
        constexpr float LOG2E = 1.4426950408889634f;
        uint32_t g = 0;
        for (int it = list_begin; it < list_end; ++it) {
            if (sh->abort_flag) break;
            const aj_task task = prm.tasks[prm.cta_ids[it]];
            const int n = task.num_kv_tiles;
            const bool store = row < task.q_rows;
            const int64_t grow = task.q_begin + row;
            const float *lse = prm.lse + ((int64_t)task.b * prm.H + task.h) * prm.Nq;
            const float *del = prm.delta + ((int64_t)task.b * prm.H + task.h) * prm.Nq;
            // dQ pass: this thread's own row (rows past the group's end are computed on neighbouring data and never stored;
            // a row without keys has lse = -inf and belongs to a task without tiles)
            float my_l2 = 0.f, my_del = 0.f;
            if (!KEYS && store) { my_l2 = lse[grow] * LOG2E; my_del = del[grow]; }
            if (!KEYS && n > 0) {
                // This thread's row of Q (warpgroup 0) or dO (warpgroup 1) as a bf16 A operand in TMEM (16 elements = 8
                // columns per MMA K step).  The previous task's MMAs are complete (its epilogue waited for them).
                const bool in = grow < prm.Na;
                const aj_tensor &src = wg ? prm.a2 : prm.a1;
                const uint4 *rowp = (const uint4 *)((const __nv_bfloat16 *)src.ptr + task.b * src.stride_b + task.h * src.stride_h + grow * src.stride_n);
#pragma unroll
                for (int half = 0; half < NB; ++half) {
                    uint32_t ra[32];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const uint4 u = in ? rowp[half * 8 + i] : make_uint4(0, 0, 0, 0);
                        ra[4 * i] = u.x; ra[4 * i + 1] = u.y; ra[4 * i + 2] = u.z; ra[4 * i + 3] = u.w;
                    }
                    tmem_st32(tmem + lane_base + (wg ? TM_A2 : TM_A1) + 32 * half, ra);
                }
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bars + 8 * BAR_A_FULL);
            }
            // Both warpgroups work on every tile: warpgroup h takes streamed rows (columns) [32 h, 32 h + 32), which halves
            // the latency between "X, Y complete" and "W, Z stored" -- with two TMEM buffers that latency, not the
            // throughput, sets the tile period.  In the KEYS pass the warpgroup whose index equals the tile's buffer
            // stages lse / delta of the tile's 64 streamed rows, fetched one of ITS tiles (two tiles) ahead.
            TileCursor cur, pf;
            cur.init(prm.r_begin, prm.r_end, task.range_begin, task.range_count);
            pf = cur;
            const int j0 = ((g & 1) != (uint32_t)wg) ? 1 : 0;      // first tile this warpgroup stages
            if (j0 == 1 && n > 1) pf.next();
            auto fetch = [&](const TileCursor &c) -> float {       // lse in log2 units (+inf past the range end: W = 0) or delta
                const int cc = st & (BC - 1);
                const bool ok = cc < c.valid();
                const int64_t qrow = c.row() + cc;
                return st < BC ? (ok ? lse[qrow] * LOG2E : INFINITY) : (ok ? del[qrow] : 0.f);
            };
            float pre = 0.f;
            if (KEYS && j0 < n) pre = fetch(pf);
            for (int j = 0; j < n; ++j, cur.next()) {
                const uint32_t gj = g + j, b = gj & 1;
                const uint32_t tX = tmem + lane_base + TM_X0 + b * TM_BUF + 32 * wg, tY = tmem + lane_base + TM_Y0 + b * TM_BUF + 32 * wg;
                const int valid = cur.valid();
                if (KEYS) {
                    if (b == (uint32_t)wg) {
                        sh->stage[b][st >> 6][st & (BC - 1)] = pre;
                        if (j + 2 < n) { pf.next(); pf.next(); pre = fetch(pf); }
                    }
                    named_bar_sync(1 + b, 256);
                }
                wait(BAR_X_FULL + b, (gj >> 1) & 1);
                tc_fence_after();
                const uint64_t sl2_2 = pack2(sl2, sl2), myl_2 = pack2(-my_l2, -my_l2), myd_2 = pack2(-my_del, -my_del);
                uint32_t xu[32], yu[32];
                tmem_ld32(tX, xu);
                tmem_ld32(tY, yu);
                tc_wait_ld(xu, yu);
                if (!KEYS && valid < BC) {                          // past the range end: S = -inf, so W = Z = 0
#pragma unroll
                    for (int c = 0; c < 32; ++c) if (32 * wg + c >= valid) xu[c] = 0xff800000u;
                }
                uint32_t wk[16], zk[16];
#pragma unroll
                for (int c4 = 0; c4 < 32; c4 += 4) {
                    uint64_t nl[2], nd[2];                          // -lse * log2e and -delta of four columns
                    if (KEYS) {
                        const float4 l4 = *reinterpret_cast<const float4 *>(&sh->stage[b][0][32 * wg + c4]);
                        const float4 d4 = *reinterpret_cast<const float4 *>(&sh->stage[b][1][32 * wg + c4]);
                        nl[0] = pack2(-l4.x, -l4.y); nl[1] = pack2(-l4.z, -l4.w);
                        nd[0] = pack2(-d4.x, -d4.y); nd[1] = pack2(-d4.z, -d4.w);
                    } else {
                        nl[0] = nl[1] = myl_2; nd[0] = nd[1] = myd_2;
                    }
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int c = c4 + 2 * h;
                        // W = exp(S - lse) = p_ab (PAPER.md:842-844 with the forward's L, :945); Z = W (dP - delta)
                        const uint64_t x = ffma2(pack2(xu[c], xu[c + 1]), sl2_2, nl[h]);
                        float x0, x1;
                        unpack2(x, x0, x1);
                        const float w0 = ex2(x0), w1 = ex2(x1);
                        const uint64_t z = fmul2(pack2(w0, w1), fadd2(pack2(yu[c], yu[c + 1]), nd[h]));
                        float z0, z1;
                        unpack2(z, z0, z1);
                        wk[c >> 1] = pack_bf16(w0, w1);
                        zk[c >> 1] = pack_bf16(z0, z1);
                    }
                }
                // bf16 W / Z over the first 16 of the 32 fp32 columns this thread has just read
                if (KEYS) tmem_st16(tX, wk);
                tmem_st16(tY, zk);
                tc_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bars + 8 * (BAR_W_FULL + b));
            }
            // ---- epilogue: acc1 * s -> dQ | dK, acc2 -> dV; each warpgroup writes one half of the D columns ----
            __nv_bfloat16 *o1 = (__nv_bfloat16 *)prm.out1.ptr + task.b * prm.out1.stride_b + task.h * prm.out1.stride_h + grow * prm.out1.stride_n;
            __nv_bfloat16 *o2 = KEYS ? (__nv_bfloat16 *)prm.out2.ptr + task.b * prm.out2.stride_b + task.h * prm.out2.stride_h + grow * prm.out2.stride_n : nullptr;
            if (n == 0) {                                           // a row without keys / a key no row sees: zeros
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = (D / 16) * wg; c < (D / 16) * (wg + 1); ++c) { ((uint4 *)o1)[c] = z; if (KEYS) ((uint4 *)o2)[c] = z; }
                }
                continue;
            }
            // A parity wait is sound only if the barrier is known to be at most one phase away: this thread consumed X of the
            // last tile, which the in-order pipe produced after the MMAs of tile n - 3 (the previous phase of that buffer's
            // barrier), and the next phase needs this thread's next hand-over.
            wait(BAR_ACC_DONE + ((g + n - 1) & 1), ((g + n - 1) >> 1) & 1);
            tc_fence_after();
            g += n;
#pragma unroll 1
            for (int cb = (D / 2) * wg; cb < (D / 2) * (wg + 1); cb += 32) {
                uint32_t a1[32], a2[32];
                tmem_ld32(tmem + lane_base + TM_ACC1 + cb, a1);
                if (KEYS) tmem_ld32(tmem + lane_base + TM_ACC2 + cb, a2);
                if (KEYS) tc_wait_ld(a1, a2); else tc_wait_ld(a1);
                if (store) {
#pragma unroll
                    for (int v4 = 0; v4 < 4; ++v4) {
                        uint32_t w1[4], w2[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int c = v4 * 8 + 2 * e;
                            w1[e] = pack_bf16(__uint_as_float(a1[c]) * prm.scale, __uint_as_float(a1[c + 1]) * prm.scale);
                            if (KEYS) w2[e] = pack_bf16(__uint_as_float(a2[c]), __uint_as_float(a2[c + 1]));
                        }
                        *(uint4 *)(o1 + cb + v4 * 8) = make_uint4(w1[0], w1[1], w1[2], w1[3]);
                        if (KEYS) *(uint4 *)(o2 + cb + v4 * 8) = make_uint4(w2[0], w2[1], w2[2], w2[3]);
                    }
                }
            }
            tc_fence_before();
            named_bar_sync(3, 256);          // the accumulators and the A columns are free only when both warpgroups are done
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    }
}

template <bool KEYS, int D>
cudaError_t launch_one(const BwdUmmaParams &prm, int grid, cudaStream_t stream, std::atomic<uint64_t> &configured) {
    if (cudaError_t e = ensure_dynamic_smem(attn_bwd_umma_kernel<KEYS, D>, (int)Cfg<D>::SMEM_TOTAL, configured)) return e;
    attn_bwd_umma_kernel<KEYS, D><<<grid, NTHREADS, Cfg<D>::SMEM_TOTAL, stream>>>(prm);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_bwd_umma(const BwdUmmaParams &prm, int d, bool keys, int grid, cudaStream_t stream) {
    if (grid <= 0 || prm.num_tasks <= 0) return cudaSuccess;
    static std::atomic<uint64_t> configured[4];
    if (d == 128) return keys ? launch_one<true, 128>(prm, grid, stream, configured[1]) : launch_one<false, 128>(prm, grid, stream, configured[0]);
    if (d == 64) return keys ? launch_one<true, 64>(prm, grid, stream, configured[3]) : launch_one<false, 64>(prm, grid, stream, configured[2]);
    return cudaErrorInvalidValue;
}

}  // namespace aj
