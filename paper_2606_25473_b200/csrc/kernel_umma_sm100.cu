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
// CTA = 8 warps, persistent, one CTA per SM:
//   warp 0      TMA producer (one lane): task fetch, Q/tQ tile, ring of {K,tK} / {V,tV} half-stages
//   warp 1      MMA issuer (one lane): QK(j+1) is issued before PV(j) so the tensor pipe never waits on softmax
//   warp 2      TMEM allocator
//   warps 4-7   softmax + tangent weights + lazy rescale + epilogue; thread = one query row (TMEM lane)
// TMEM columns (fp32): O [0,128) | T [128,256) | S0 [256,320) tS0 [320,384) | S1 [384,448) tS1 [448,512);
// P~ and H~ (bf16, 32 columns each) overwrite the first half of their S / tS buffer.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

#include "kernels.hpp"

namespace aj {

namespace {

constexpr int BR = UMMA_TILE_Q;        // 128 query rows
constexpr int BC = UMMA_TILE_K;        // 64 keys per tile
constexpr int D = 128;
constexpr int NSTAGE = 5;              // ring slots of 32 KB ({K,tK} or {V,tV} of one tile)
constexpr uint32_t Q_BYTES = BR * D * 2;           // 32 KB
constexpr uint32_t QHALF_BYTES = BR * 64 * 2;      // one 64-column swizzle block of Q: 16 KB
constexpr uint32_t KV_BYTES = BC * D * 2;          // 16 KB
constexpr uint32_t KVHALF_BYTES = BC * 64 * 2;     // 8 KB
constexpr uint32_t SLOT_BYTES = 2 * KV_BYTES;      // 32 KB
constexpr uint32_t SMEM_TILES = 2 * Q_BYTES + NSTAGE * SLOT_BYTES;  // 224 KB
constexpr uint32_t SMEM_TOTAL = SMEM_TILES + 1024 /*align*/ + 256 /*barriers*/;
constexpr int NTHREADS = 256;

constexpr uint32_t TM_O = 0, TM_T = 128, TM_S0 = 256, TM_TS0 = 320, TM_SBUF = 128;  // S1 = S0 + 128, ...
constexpr float RESCALE_THRESHOLD = 8.0f;  // log2 units

// Barrier indices inside the shared barrier array.
enum {
    BAR_Q_FULL = 0, BAR_Q_EMPTY,
    BAR_KV_FULL, BAR_KV_EMPTY = BAR_KV_FULL + NSTAGE,
    BAR_S_FULL = BAR_KV_EMPTY + NSTAGE, BAR_P_FULL = BAR_S_FULL + 2, BAR_PV_DONE = BAR_P_FULL + 2,
    BAR_TASK_FULL = BAR_PV_DONE + 2, BAR_TASK_EMPTY = BAR_TASK_FULL + 2, NUM_BARS = BAR_TASK_EMPTY + 2
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier -------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug prints where it is stuck and makes every role leave instead of hanging the GPU.
__device__ __forceinline__ bool mbar_wait(uint32_t bar0, int idx, uint32_t parity, volatile int *abort_flag) {
    const uint32_t bar = bar0 + 8u * idx;
    if (mbar_try_wait(bar, parity)) return true;
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++spins & 0xff) == 0) {
            if (*abort_flag) return false;
            if (clock64() - t0 > 4000000000LL) {
                printf("attn_jvp umma: timeout block %d thread %d barrier %d parity %u\n", blockIdx.x, threadIdx.x, idx, parity);
                *abort_flag = 1;
                return false;
            }
        }
    }
    return true;
}

// ---- TMA ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap *map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// ---- tcgen05 --------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accum) : "memory");
}

#define AJ_R8(r, o) "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), "=r"(r[o + 5]), "=r"(r[o + 6]), "=r"(r[o + 7])
#define AJ_I8(r, o) "r"(r[o + 0]), "r"(r[o + 1]), "r"(r[o + 2]), "r"(r[o + 3]), "r"(r[o + 4]), "r"(r[o + 5]), "r"(r[o + 6]), "r"(r[o + 7])

// 32 lanes x 32 consecutive fp32 columns: thread t of the warp gets lane (taddr.lane + t).
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : AJ_R8(r, 0), AJ_R8(r, 8), AJ_R8(r, 16), AJ_R8(r, 24) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%32], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31};"
        ::AJ_I8(r, 0), AJ_I8(r, 8), AJ_I8(r, 16), AJ_I8(r, 24), "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%16], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15};"
        ::AJ_I8(r, 0), AJ_I8(r, 8), "r"(taddr) : "memory");
}

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// bf16x2 with `lo` in bits [0,16) and `hi` in bits [16,32), round to nearest even
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// Shared-memory matrix descriptors (PTX ISA "tcgen05 shared memory descriptor"): start address, leading / stride
// byte offsets in 16-byte units, descriptor version 1 (bit 46), 128-byte swizzle (value 2 in bits 61-63).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor for kind::f16: D fp32 (bits 4-5 = 1), A and B bf16 (bits 7-9, 10-12 = 1), B major (bit 16),
// N >> 3 (bits 17-22), M >> 4 (bits 24-28).
constexpr uint32_t make_idesc(int n, bool b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(BR >> 4) << 24);
}
constexpr uint32_t IDESC_QK = make_idesc(BC, false);  // 128 x 64 x 16, A and B K-major
constexpr uint32_t IDESC_PV = make_idesc(D, true);    // 128 x 128 x 16, A from TMEM, B (V) MN-major

// Walks the key tiles of a task in order: ranges [rb, rb + rc), each cut into BC-key tiles from its start.
struct TileCursor {
    const int32_t *kb, *ke;
    int r, rend, k, kend;
    __device__ void init(const int32_t *k_begin, const int32_t *k_end, int rb, int rc) {
        kb = k_begin; ke = k_end; r = rb; rend = rb + rc;
        if (r < rend) { k = kb[r]; kend = ke[r]; } else { k = 0; kend = 0; }
    }
    __device__ int key_row() const { return k; }
    __device__ int valid() const { return min(BC, kend - k); }
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

__global__ void __launch_bounds__(NTHREADS, 1)
attn_jvp_umma_kernel(const __grid_constant__ UmmaParams prm) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t tiles = (raw + 1023u) & ~1023u;       // 1024-byte alignment for the 128-byte swizzle
    Shared *sh = reinterpret_cast<Shared *>(smem_raw + (tiles - raw) + SMEM_TILES);
    const uint32_t sQ = tiles, sTQ = tiles + Q_BYTES, sRing = tiles + 2 * Q_BYTES;
    const uint32_t bars = smem_u32(sh->bars);
    volatile int *abort_flag = &sh->abort_flag;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        mbar_init(bars + 8 * BAR_Q_FULL, 1);
        mbar_init(bars + 8 * BAR_Q_EMPTY, 1);
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bars + 8 * (BAR_KV_FULL + i), 1); mbar_init(bars + 8 * (BAR_KV_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bars + 8 * (BAR_S_FULL + i), 1);
            mbar_init(bars + 8 * (BAR_P_FULL + i), 128);
            mbar_init(bars + 8 * (BAR_PV_DONE + i), 1);
            mbar_init(bars + 8 * (BAR_TASK_FULL + i), 1);
            mbar_init(bars + 8 * (BAR_TASK_EMPTY + i), 5);   // MMA lane + one lane of each softmax warp
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
            int task_id = blockIdx.x;
            for (uint32_t t = 0;; ++t) {
                const int ts = t & 1;
                if (!mbar_wait(bars, BAR_TASK_EMPTY + ts, ((t >> 1) & 1) ^ 1, abort_flag)) break;
                sh->task_id[ts] = task_id;
                mbar_arrive(bars + 8 * (BAR_TASK_FULL + ts));
                if (task_id >= prm.num_tasks) break;
                const aj_task task = prm.tasks[task_id];
                task_id = atomicAdd(&prm.counters[0], 1) + gridDim.x;
                if (task.num_kv_tiles == 0) continue;
                // Q_i, tQ_i: two 64-column swizzle blocks each
                if (!mbar_wait(bars, BAR_Q_EMPTY, (nq & 1) ^ 1, abort_flag)) break;
                mbar_expect_tx(bars + 8 * BAR_Q_FULL, 2 * Q_BYTES);
                tma_load_4d(sQ, &prm.tm_q, bars + 8 * BAR_Q_FULL, 0, task.q_begin, task.h, task.b);
                tma_load_4d(sQ + QHALF_BYTES, &prm.tm_q, bars + 8 * BAR_Q_FULL, 64, task.q_begin, task.h, task.b);
                tma_load_4d(sTQ, &prm.tm_tq, bars + 8 * BAR_Q_FULL, 0, task.q_begin, task.h, task.b);
                tma_load_4d(sTQ + QHALF_BYTES, &prm.tm_tq, bars + 8 * BAR_Q_FULL, 64, task.q_begin, task.h, task.b);
                ++nq;
                // ring order = MMA consumption order: KtK(0), KtK(1), VtV(0), KtK(2), VtV(1), ...
                TileCursor ck, cv;
                ck.init(prm.k_begin, prm.k_end, task.range_begin, task.range_count);
                cv = ck;
                const int n = task.num_kv_tiles;
                auto push = [&](bool is_k) -> bool {
                    const uint32_t slot = ring % NSTAGE;
                    if (!mbar_wait(bars, BAR_KV_EMPTY + slot, ((ring / NSTAGE) & 1) ^ 1, abort_flag)) return false;
                    const uint32_t dst = sRing + slot * SLOT_BYTES, full = bars + 8 * (BAR_KV_FULL + slot);
                    mbar_expect_tx(full, SLOT_BYTES);
                    TileCursor &c = is_k ? ck : cv;
                    const CUtensorMap *m0 = is_k ? &prm.tm_k : &prm.tm_v, *m1 = is_k ? &prm.tm_tk : &prm.tm_tv;
                    const int row = c.key_row();
                    tma_load_4d(dst, m0, full, 0, row, task.h, task.b);
                    tma_load_4d(dst + KVHALF_BYTES, m0, full, 64, row, task.h, task.b);
                    tma_load_4d(dst + KV_BYTES, m1, full, 0, row, task.h, task.b);
                    tma_load_4d(dst + KV_BYTES + KVHALF_BYTES, m1, full, 64, row, task.h, task.b);
                    c.next();
                    ++ring;
                    return true;
                };
                bool ok = push(true);
                for (int j = 0; j < n && ok; ++j) {
                    if (j + 1 < n) ok = push(true);
                    if (ok) ok = push(false);
                }
                if (!ok) break;
            }
            // the last CTA to run out of work re-arms the counters for the next launch
            if (!*abort_flag) {
                const int done = atomicAdd(&prm.counters[1], 1);
                if (done == (int)gridDim.x - 1) { prm.counters[0] = 0; prm.counters[1] = 0; __threadfence(); }
            }
        }
    } else if (warp == 1) {
        // ================================================= MMA issuer ============================================
        if (lane == 0) {
            uint32_t ring = 0, nq = 0, g = 0;   // g = tiles issued so far (selects S/tS buffer and barrier phase)
            for (uint32_t t = 0;; ++t) {
                const int ts = t & 1;
                if (!mbar_wait(bars, BAR_TASK_FULL + ts, (t >> 1) & 1, abort_flag)) break;
                const int task_id = sh->task_id[ts];
                mbar_arrive(bars + 8 * (BAR_TASK_EMPTY + ts));
                if (task_id >= prm.num_tasks) break;
                const int n = prm.tasks[task_id].num_kv_tiles;
                if (n == 0) continue;
                if (!mbar_wait(bars, BAR_Q_FULL, nq & 1, abort_flag)) break;
                ++nq;
                tc_fence_after();
                bool ok = true;
                auto issue_qk = [&](uint32_t gj) -> bool {
                    const uint32_t slot = ring % NSTAGE;
                    if (!mbar_wait(bars, BAR_KV_FULL + slot, (ring / NSTAGE) & 1, abort_flag)) return false;
                    tc_fence_after();
                    const uint32_t sK = sRing + slot * SLOT_BYTES, sTK = sK + KV_BYTES;
                    const uint32_t tS_ = tmem + TM_S0 + (gj & 1) * TM_SBUF, tTS_ = tmem + TM_TS0 + (gj & 1) * TM_SBUF;
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t qoff = (ks >> 2) * QHALF_BYTES + (ks & 3) * 32;
                        const uint32_t koff = (ks >> 2) * KVHALF_BYTES + (ks & 3) * 32;
                        const uint64_t dq = make_desc(sQ + qoff, 16, 1024), dtq = make_desc(sTQ + qoff, 16, 1024);
                        const uint64_t dk = make_desc(sK + koff, 16, 1024), dtk = make_desc(sTK + koff, 16, 1024);
                        mma_ss(tS_, dq, dk, IDESC_QK, ks > 0);        // S  = Q K^T
                        mma_ss(tTS_, dtq, dk, IDESC_QK, ks > 0);      // tS = tQ K^T
                        mma_ss(tTS_, dq, dtk, IDESC_QK, 1);           //    + Q tK^T
                    }
                    tc_commit(bars + 8 * (BAR_KV_EMPTY + slot));
                    tc_commit(bars + 8 * (BAR_S_FULL + (gj & 1)));
                    ++ring;
                    return true;
                };
                if (!issue_qk(g)) break;
                for (int j = 0; j < n; ++j) {
                    const uint32_t gj = g + j;
                    if (j + 1 < n) { if (!issue_qk(gj + 1)) { ok = false; break; } }
                    else tc_commit(bars + 8 * BAR_Q_EMPTY);           // every QK of this task has been issued
                    if (!mbar_wait(bars, BAR_P_FULL + (gj & 1), (gj >> 1) & 1, abort_flag)) { ok = false; break; }
                    const uint32_t slot = ring % NSTAGE;
                    if (!mbar_wait(bars, BAR_KV_FULL + slot, (ring / NSTAGE) & 1, abort_flag)) { ok = false; break; }
                    tc_fence_after();
                    const uint32_t sV = sRing + slot * SLOT_BYTES, sTV = sV + KV_BYTES;
                    const uint32_t tP = tmem + TM_S0 + (gj & 1) * TM_SBUF, tH = tmem + TM_TS0 + (gj & 1) * TM_SBUF;
#pragma unroll
                    for (int ks = 0; ks < BC / 16; ++ks) {
                        // V tile in smem: key row r at r*128 bytes inside each 64-column block; blocks 8 KB apart.
                        const uint64_t dv = make_desc(sV + ks * 2048, KVHALF_BYTES, 1024);
                        const uint64_t dtv = make_desc(sTV + ks * 2048, KVHALF_BYTES, 1024);
                        const uint32_t acc = (j > 0 || ks > 0) ? 1u : 0u;
                        mma_ts(tmem + TM_O, tP + ks * 8, dv, IDESC_PV, acc);     // O += P~ V
                        mma_ts(tmem + TM_T, tP + ks * 8, dtv, IDESC_PV, acc);    // T += P~ tV
                        mma_ts(tmem + TM_T, tH + ks * 8, dv, IDESC_PV, 1);       // T += H~ V
                    }
                    tc_commit(bars + 8 * (BAR_KV_EMPTY + slot));
                    tc_commit(bars + 8 * (BAR_PV_DONE + (gj & 1)));
                    ++ring;
                }
                if (!ok) break;
                g += n;
            }
        }
    } else if (warp >= 4) {
        // ================================================= softmax / tangent weights / epilogue ==================
        const int row = threadIdx.x - 128;                       // query row inside the tile = TMEM lane
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const float sl2 = prm.scale_log2, sc = prm.scale;
        uint32_t g = 0;
        for (uint32_t t = 0;; ++t) {
            const int ts = t & 1;
            if (!mbar_wait(bars, BAR_TASK_FULL + ts, (t >> 1) & 1, abort_flag)) break;
            const int task_id = sh->task_id[ts];
            __syncwarp();
            if (lane == 0) mbar_arrive(bars + 8 * (BAR_TASK_EMPTY + ts));
            if (task_id >= prm.num_tasks) break;
            const aj_task task = prm.tasks[task_id];
            const int n = task.num_kv_tiles;
            float m_ref = 0.f, l = 0.f, r = 0.f;
            TileCursor cur;
            cur.init(prm.k_begin, prm.k_end, task.range_begin, task.range_count);
            bool ok = true;
            for (int j = 0; j < n; ++j, cur.next()) {
                const uint32_t gj = g + j, b = gj & 1;
                const uint32_t tS_ = tmem + lane_base + TM_S0 + b * TM_SBUF, tTS_ = tmem + lane_base + TM_TS0 + b * TM_SBUF;
                if (!mbar_wait(bars, BAR_S_FULL + b, (gj >> 1) & 1, abort_flag)) { ok = false; break; }
                tc_fence_after();
                uint32_t su[2][32];
                tmem_ld32(tS_, su[0]);
                tmem_ld32(tS_ + 32, su[1]);
                tc_wait_ld();
                float s[BC];
#pragma unroll
                for (int c = 0; c < BC; ++c) s[c] = __uint_as_float(su[c >> 5][c & 31]);
                const int valid = cur.valid();
                if (valid < BC) {                                 // tile-valid mask: S = -inf
#pragma unroll
                    for (int c = 0; c < BC; ++c) if (c >= valid) s[c] = -INFINITY;
                }
                float mx = s[0];
#pragma unroll
                for (int c = 1; c < BC; ++c) mx = fmaxf(mx, s[c]);
                const float cand = mx * sl2;
                if (j == 0) {
                    m_ref = cand;
                } else {
                    const bool need = cand > m_ref + RESCALE_THRESHOLD;
                    if (__any_sync(0xffffffffu, need)) {
                        // e^{m - m_new} applied to O, T (= A + B), l, r; needs PV(j-1) finished
                        const uint32_t gp = gj - 1;
                        if (!mbar_wait(bars, BAR_PV_DONE + (gp & 1), (gp >> 1) & 1, abort_flag)) { ok = false; break; }
                        tc_fence_after();
                        const float f = need ? ex2(m_ref - cand) : 1.f;
#pragma unroll 1
                        for (int cb = 0; cb < 256; cb += 32) {
                            uint32_t a[32];
                            tmem_ld32(tmem + lane_base + cb, a);
                            tc_wait_ld();
#pragma unroll
                            for (int c = 0; c < 32; ++c) a[c] = __float_as_uint(__uint_as_float(a[c]) * f);
                            tmem_st32(tmem + lane_base + cb, a);
                        }
                        l *= f; r *= f;
                        if (need) m_ref = cand;
                    }
                }
                // P~ = exp2(S*s*log2e - m_ref); l += rowsum
#pragma unroll
                for (int c = 0; c < BC; ++c) { s[c] = ex2(fmaf(s[c], sl2, -m_ref)); l += s[c]; }
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    uint32_t pk[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) pk[c] = pack_bf16(s[hh * 32 + 2 * c], s[hh * 32 + 2 * c + 1]);
                    tmem_st16(tS_ + hh * 16, pk);
                }
                // H~ = P~ o (s * tS); r += rowsum.  Masked columns have P~ = 0, so H~ = 0.
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    uint32_t tu[32];
                    tmem_ld32(tTS_ + hh * 32, tu);
                    tc_wait_ld();
                    uint32_t pk[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) {
                        const float h0 = s[hh * 32 + 2 * c] * (__uint_as_float(tu[2 * c]) * sc);
                        const float h1 = s[hh * 32 + 2 * c + 1] * (__uint_as_float(tu[2 * c + 1]) * sc);
                        r += h0; r += h1;
                        pk[c] = pack_bf16(h0, h1);
                    }
                    tmem_st16(tTS_ + hh * 16, pk);
                }
                tc_wait_st();
                tc_fence_before();
                mbar_arrive(bars + 8 * (BAR_P_FULL + b));
            }
            if (!ok) break;
            // ---- epilogue (Eq. 45) ----
            const bool store = row < task.q_rows;
            const int64_t grow = task.q_begin + row;
            __nv_bfloat16 *op = (__nv_bfloat16 *)prm.o.ptr + task.b * prm.o.stride_b + task.h * prm.o.stride_h + grow * prm.o.stride_n;
            __nv_bfloat16 *tp = (__nv_bfloat16 *)prm.to.ptr + task.b * prm.to.stride_b + task.h * prm.to.stride_h + grow * prm.to.stride_n;
            if (n == 0) {                                         // no key: O = 0, tO = 0, lse = -inf (R9)
                if (store) {
                    const uint4 z = make_uint4(0, 0, 0, 0);
                    for (int c = 0; c < D / 8; ++c) { ((uint4 *)op)[c] = z; ((uint4 *)tp)[c] = z; }
                    if (prm.lse) prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = -INFINITY;
                }
                continue;
            }
            {
                const uint32_t gl = g + n - 1;
                if (!mbar_wait(bars, BAR_PV_DONE + (gl & 1), (gl >> 1) & 1, abort_flag)) break;
                tc_fence_after();
            }
            const float inv = 1.f / l, rl = r * inv;
#pragma unroll 1
            for (int cb = 0; cb < D; cb += 32) {
                uint32_t ao[32], at[32];
                tmem_ld32(tmem + lane_base + TM_O + cb, ao);
                tmem_ld32(tmem + lane_base + TM_T + cb, at);
                tc_wait_ld();
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
            if (store && prm.lse)
                prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + grow] = (m_ref + log2f(l)) * 0.6931471805599453f;
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

size_t umma_smem_bytes() { return SMEM_TOTAL; }

cudaError_t launch_umma(const UmmaParams &prm, int grid, cudaStream_t stream) {
    if (grid <= 0) return cudaSuccess;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(attn_jvp_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_TOTAL);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    attn_jvp_umma_kernel<<<grid, NTHREADS, SMEM_TOTAL, stream>>>(prm);
    return cudaGetLastError();
}

}  // namespace aj
