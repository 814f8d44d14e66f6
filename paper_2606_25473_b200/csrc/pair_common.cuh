// Pieces shared by the CTA-pair tcgen05 kernels (forward + JVP, primal backward): bounded barrier waits and the cursors
// that walk a task's schedule entries in 64-row tiles.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

#include "kernels.hpp"
#include "umma_ptx.cuh"

namespace aj {
namespace pairk {

constexpr int BC = UMMA_TILE_K;        // 64 streamed rows (keys in the forward) per tile

// Bounded wait (see ptx::Waiter): after ~2 s the waiter reports where it is stuck, raises the CTA's abort flag and the
// plan's error word; from then on every wait of the CTA returns at once and all roles run off the end of their work.
static __device__ __noinline__ void pair_wait_slow(uint32_t bar, int idx, uint32_t parity, volatile int *abort_flag, int32_t *err, int code_base) {
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (!ptx::mbar_try_wait(bar, parity)) {
        if ((++spins & 0x3f) == 0) {
            if (*abort_flag) return;
            if (clock64() - t0 > 4000000000LL) {
                printf("attn_jvp pair kernel %d: timeout block %d thread %d barrier %d parity %u\n", code_base, blockIdx.x, threadIdx.x, idx, parity);
                *abort_flag = 1;
                atomicExch(err, code_base + idx);
                return;
            }
        }
    }
}
struct PairWaiter {
    uint32_t bars;
    volatile int *abort_flag;
    int32_t *err;
    int code_base;       // 100: forward, 200 / 300: backward dQ / dK,dV pass
    __device__ __forceinline__ void operator()(int idx, uint32_t parity) const {
        const uint32_t bar = bars + 8u * idx;
        if (ptx::mbar_try_wait(bar, parity)) return;
        if (ptx::mbar_try_wait(bar, parity)) return;
        pair_wait_slow(bar, idx, parity, abort_flag, err, code_base);
    }
};

// The same bounded wait without a function call and without printf, for roles that run under a raised register budget
// (setmaxnreg): a call in such a region makes ptxas spill everything that is live across it.
struct PairWaiterInline {
    uint32_t bars;
    volatile int *abort_flag;
    int32_t *err;
    int code_base;
    __device__ __forceinline__ void operator()(int idx, uint32_t parity) const {
        const uint32_t bar = bars + 8u * idx;
        if (ptx::mbar_try_wait(bar, parity)) return;
        const long long t0 = clock64();
        uint32_t spins = 0;
        while (!ptx::mbar_try_wait(bar, parity)) {
            if ((++spins & 0x3f) == 0) {
                if (*abort_flag) return;
                if (clock64() - t0 > 4000000000LL) { *abort_flag = 1; atomicExch(err, code_base + idx); return; }
            }
        }
    }
};

// One 64-row tile of a task's stream.
struct Tile { int key_row, valid, entry; };
// Walks the streamed tiles of a task in order: schedule entries [rb, rb + rc), each cut into BC-row tiles from its start.
struct TileCursor {
    const int32_t *kb, *ke;
    int r, rend, k, kend;
    __device__ void init(const int32_t *k_begin, const int32_t *k_end, int rb, int rc) {
        kb = k_begin; ke = k_end; r = rb; rend = rb + rc;
        if (r < rend) { k = kb[r]; kend = ke[r]; } else { k = 0; kend = 0; }
    }
    __device__ Tile get() const { return Tile{k, min(BC, kend - k), r}; }
    __device__ void next() {
        k += BC;
        if (k >= kend) { ++r; if (r < rend) { k = kb[r]; kend = ke[r]; } }
    }
};

// A stationary row's view of a task's stream: how many columns of the next tile this thread's row sees (PAPER.md:909-914:
// inside the entry's range and the entry's row interval).  The next entry is fetched when the current one is entered,
// so that crossing into it costs no memory latency.
struct RowCursor {
    const int32_t *kb, *ke;
    const uint32_t *rows;
    int r, rend, prow;
    int rem;             // streamed rows left in the current entry
    bool sees;           // this row is inside the current entry's row interval
    int nkb, nke;        // the next entry as loaded (decoded only when it is entered, so the loads stay in flight)
    uint32_t nrr;
    __device__ __forceinline__ void fetch_next() {
        if (r + 1 < rend) { nkb = kb[r + 1]; nke = ke[r + 1]; nrr = rows[r + 1]; }
        else { nkb = 0; nke = 0; nrr = 0; }
    }
    __device__ __forceinline__ void advance() {
        ++r;
        rem = nke - nkb;
        sees = prow >= (int)(nrr & 0xffffu) && prow < (int)((nrr >> 16) & 0x7fffu);
        fetch_next();
    }
    __device__ __forceinline__ void init(const int32_t *k_begin, const int32_t *k_end, const uint32_t *row_iv, int rb, int rc, int row) {
        kb = k_begin; ke = k_end; rows = row_iv; r = rb - 2; rend = rb + rc; prow = row;
        nkb = 0; nke = 0; nrr = 0;
        advance();           // r = rb - 1: fetches entry rb
        advance();           // r = rb: current = entry rb, next = entry rb + 1
    }
    // columns of the next tile this row sees; consumes the tile
    __device__ __forceinline__ int tile() {
        const int v = sees ? min(BC, rem) : 0;
        rem -= BC;
        if (rem <= 0) advance();
        return v;
    }
    // both tiles of a pair-step that lies inside the current entry
    __device__ __forceinline__ bool pair_inside() const { return rem >= 2 * BC; }
    __device__ __forceinline__ int pair() {
        const int v = sees ? BC : 0;
        rem -= 2 * BC;
        if (rem <= 0) advance();
        return v;
    }
};

}  // namespace pairk
}  // namespace aj
