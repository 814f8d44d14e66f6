// Plain-FMA fp32 attention + JVP kernel (the fp32-input path; also runs bf16 inputs for debugging).
//
// One CTA per task = one tile of TQ query rows inside one query group; it streams the task's key ranges in
// tiles of TK keys and follows Algorithm 1 of the paper line by line: scores and score
// tangents (Eq. 42-43, scaled, R1), tile-valid mask (S = -inf, tS = 0), running max / l / r,
// rescale of O, A, B (kept merged as T = A + B), the three accumulations, and the epilogue
// O/l, L = m + log l, tO = (T - r O)/l (Eq. 45).  All arithmetic is fp32 FMA; no TF32 (R14).
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include "kernels.hpp"

namespace aj {

namespace {

constexpr int TQ = SIMT_TILE_Q;  // query rows per CTA
constexpr int TK = SIMT_TILE_K;  // keys per tile (= warp width: one key per lane)
constexpr int NWARPS = 4;
constexpr int ROWS_PER_WARP = TQ / NWARPS;

template <typename T> __device__ __forceinline__ float to_f32(T x);
template <> __device__ __forceinline__ float to_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f32(float x);
template <> __device__ __forceinline__ float from_f32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

__device__ __forceinline__ float warp_max(float x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmaxf(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
}
__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// PRIMAL: a plan without tangents (AJ_TANGENT_NONE): tq, tk, tv are never read (they may be NULL), tO = 0, tlse = 0.
template <typename T, int D, bool PRIMAL>
__global__ void __launch_bounds__(NWARPS * 32)
attn_jvp_simt_kernel(SimtParams prm) {
    constexpr int DP = D + 1;        // padded row: lane-per-key reads hit distinct banks
    constexpr int DL = D / 32;       // output dims owned by a lane
    extern __shared__ float smem[];
    float *sQ = smem;                // [TQ][D]
    float *sTQ = sQ + TQ * D;        // [TQ][D]
    float *sK = sTQ + TQ * D;        // [TK][DP]
    float *sTK = sK + TK * DP;
    float *sV = sTK + TK * DP;
    float *sTV = sV + TK * DP;

    const aj_task task = prm.tasks[blockIdx.x];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const T *q = (const T *)prm.q.ptr + task.b * prm.q.stride_b + task.h * prm.q.stride_h;
    const T *tq = PRIMAL ? nullptr : (const T *)prm.tq.ptr + task.b * prm.tq.stride_b + task.h * prm.tq.stride_h;
    const T *k = (const T *)prm.k.ptr + task.b * prm.k.stride_b + task.h * prm.k.stride_h;
    const T *tk = PRIMAL ? nullptr : (const T *)prm.tk.ptr + task.b * prm.tk.stride_b + task.h * prm.tk.stride_h;
    const T *v = (const T *)prm.v.ptr + task.b * prm.v.stride_b + task.h * prm.v.stride_h;
    const T *tv = PRIMAL ? nullptr : (const T *)prm.tv.ptr + task.b * prm.tv.stride_b + task.h * prm.tv.stride_h;

    // Alg. 1 line "Load Q_i, tQ_i"; rows past the group end are zero and never stored.
    for (int i = threadIdx.x; i < TQ * D; i += blockDim.x) {
        int r = i / D, c = i % D;
        bool ok = r < task.q_rows;
        sQ[i] = ok ? to_f32(q[(int64_t)(task.q_begin + r) * prm.q.stride_n + c]) : 0.f;
        sTQ[i] = (ok && !PRIMAL) ? to_f32(tq[(int64_t)(task.q_begin + r) * prm.tq.stride_n + c]) : 0.f;
    }

    float m[ROWS_PER_WARP], l[ROWS_PER_WARP], rs[ROWS_PER_WARP];
    float accO[ROWS_PER_WARP][DL], accT[ROWS_PER_WARP][DL];
#pragma unroll
    for (int i = 0; i < ROWS_PER_WARP; ++i) {
        m[i] = -CUDART_INF_F; l[i] = 0.f; rs[i] = 0.f;
#pragma unroll
        for (int j = 0; j < DL; ++j) { accO[i][j] = 0.f; accT[i][j] = 0.f; }
    }

    for (int ri = 0; ri < task.range_count; ++ri) {          // PAPER.md:903 each allowed key range
        const int k0 = prm.k_begin[task.range_begin + ri], k1 = prm.k_end[task.range_begin + ri];
        for (int kt = k0; kt < k1; kt += TK) {               // PAPER.md:905 each key/value tile
            __syncthreads();
            for (int i = threadIdx.x; i < TK * D; i += blockDim.x) {
                int r = i / D, c = i % D;
                bool ok = kt + r < k1;
                int64_t row = kt + r;
                sK[r * DP + c] = ok ? to_f32(k[row * prm.k.stride_n + c]) : 0.f;
                sTK[r * DP + c] = (ok && !PRIMAL) ? to_f32(tk[row * prm.tk.stride_n + c]) : 0.f;
                sV[r * DP + c] = ok ? to_f32(v[row * prm.v.stride_n + c]) : 0.f;
                sTV[r * DP + c] = (ok && !PRIMAL) ? to_f32(tv[row * prm.tv.stride_n + c]) : 0.f;
            }
            __syncthreads();
            const bool valid = kt + lane < k1;               // tile-valid mask B_ij
#pragma unroll
            for (int i = 0; i < ROWS_PER_WARP; ++i) {
                const int r = warp * ROWS_PER_WARP + i;
                const float *qr = sQ + r * D, *tqr = sTQ + r * D;
                const float *kc = sK + lane * DP, *tkc = sTK + lane * DP;
                float s = 0.f, ts = 0.f;
#pragma unroll 8
                for (int c = 0; c < D; ++c) {
                    s = fmaf(qr[c], kc[c], s);
                    ts = fmaf(tqr[c], kc[c], ts);
                    ts = fmaf(qr[c], tkc[c], ts);
                }
                s = valid ? s * prm.scale : -CUDART_INF_F;
                ts = valid ? ts * prm.scale : 0.f;
                const float m_new = fmaxf(m[i], warp_max(s));
                const float p = valid ? expf(s - m_new) : 0.f;
                const float hh = p * ts;
                const float alpha = expf(m[i] - m_new);                // e^{m - m_new}; 0 on the first tile
                l[i] = alpha * l[i] + warp_sum(p);
                rs[i] = alpha * rs[i] + warp_sum(hh);
                m[i] = m_new;
#pragma unroll
                for (int j = 0; j < DL; ++j) { accO[i][j] *= alpha; accT[i][j] *= alpha; }
                for (int c = 0; c < TK; ++c) {
                    const float pc = __shfl_sync(0xffffffffu, p, c);
                    const float hc = __shfl_sync(0xffffffffu, hh, c);
#pragma unroll
                    for (int j = 0; j < DL; ++j) {
                        const float vv = sV[c * DP + lane + 32 * j];
                        const float tvv = sTV[c * DP + lane + 32 * j];
                        accO[i][j] = fmaf(pc, vv, accO[i][j]);                       // O += P V      (:928)
                        accT[i][j] = fmaf(pc, tvv, fmaf(hc, vv, accT[i][j]));         // A + B merged (:930,:937)
                    }
                }
            }
        }
    }

    // Epilogue.  A task with no keys writes O = 0, tO = 0, lse = -inf (R9).
    T *o = (T *)prm.o.ptr + task.b * prm.o.stride_b + task.h * prm.o.stride_h;
    T *to = prm.to.ptr ? (T *)prm.to.ptr + task.b * prm.to.stride_b + task.h * prm.to.stride_h : nullptr;
#pragma unroll
    for (int i = 0; i < ROWS_PER_WARP; ++i) {
        const int r = warp * ROWS_PER_WARP + i;
        if (r >= task.q_rows) continue;
        const int64_t row = task.q_begin + r;
        const bool empty = !(l[i] > 0.f);
        const float inv = empty ? 0.f : 1.f / l[i];
        const float rl = rs[i] * inv;
#pragma unroll
        for (int j = 0; j < DL; ++j) {
            const float on = accO[i][j] * inv;
            const float tn = accT[i][j] * inv - rl * on;             // Eq. 45
            o[row * prm.o.stride_n + lane + 32 * j] = from_f32<T>(on);
            if (to) to[row * prm.to.stride_n + lane + 32 * j] = from_f32<T>(PRIMAL ? 0.f : tn);
        }
        if (prm.lse && lane == 0)
            prm.lse[((int64_t)task.b * prm.H + task.h) * prm.Nq + row] = empty ? -CUDART_INF_F : m[i] + logf(l[i]);
        if (prm.tlse && lane == 0)                                    // tangent of lse: r / l
            prm.tlse[((int64_t)task.b * prm.H + task.h) * prm.Nq + row] = PRIMAL ? 0.f : rl;
    }
}

template <typename T, int D, bool PRIMAL>
cudaError_t launch_p(const SimtParams &prm, int num_tasks, cudaStream_t stream) {
    const size_t smem = sizeof(float) * (2 * TQ * D + 4 * TK * (D + 1));
    static std::atomic<uint64_t> configured{0};
    if (cudaError_t e = ensure_dynamic_smem(attn_jvp_simt_kernel<T, D, PRIMAL>, (int)smem, configured)) return e;
    attn_jvp_simt_kernel<T, D, PRIMAL><<<num_tasks, NWARPS * 32, smem, stream>>>(prm);
    return cudaGetLastError();
}
template <typename T, int D>
cudaError_t launch_t(const SimtParams &prm, int num_tasks, cudaStream_t stream) {
    return prm.no_tangents ? launch_p<T, D, true>(prm, num_tasks, stream) : launch_p<T, D, false>(prm, num_tasks, stream);
}

}  // namespace

cudaError_t launch_simt(const SimtParams &prm, int dtype, int d, int num_tasks, cudaStream_t stream) {
    if (num_tasks == 0) return cudaSuccess;
    if (dtype == AJ_FP32 && d == 64) return launch_t<float, 64>(prm, num_tasks, stream);
    if (dtype == AJ_FP32 && d == 128) return launch_t<float, 128>(prm, num_tasks, stream);
    if (dtype == AJ_BF16 && d == 64) return launch_t<__nv_bfloat16, 64>(prm, num_tasks, stream);
    if (dtype == AJ_BF16 && d == 128) return launch_t<__nv_bfloat16, 128>(prm, num_tasks, stream);
    return cudaErrorInvalidValue;
}

}  // namespace aj
