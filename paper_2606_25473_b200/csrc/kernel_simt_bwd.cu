// Primal backward of masked attention: dQ, dK, dV from dO, O and lse -- plain-FMA fp32 kernels.
//
// The student's gradient flows through the ordinary primal path (Eq. 19) and the forward returns
// L = lse for it.  With P = exp(S - lse) recomputed tile by tile (S = scale Q K^T, masked entries 0):
//     delta_a = <dO_a, O_a>                  (= sum_b p_ab dP_ab, because O_a = sum_b p_ab v_b)
//     dP_ab = <dO_a, v_b>,  dS_ab = p_ab (dP_ab - delta_a)
//     dQ_a = scale sum_b dS_ab k_b          one CTA per query tile, streaming the key ranges of its group
//     dV_b = sum_a p_ab dO_a,  dK_b = scale sum_a dS_ab q_a      one CTA per KEY tile, streaming the row ranges that
//                                                                  see it (the transposed schedule), so no atomics
// These kernels serve fp32 inputs, d = 64 and plans forced to AJ_KERNEL_SIMT (fp32 arithmetic for both input dtypes), and
// the delta kernel serves both backward paths; bf16 with d = 128 runs kernel_umma_bwd_sm100.cu (tcgen05).
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include "kernels.hpp"

namespace aj {

namespace {

constexpr int TS = SIMT_TILE_Q;  // stationary rows per CTA (query rows for dQ, keys for dK/dV)
constexpr int TM = SIMT_TILE_K;  // streamed rows per tile (= warp width: one streamed row per lane)
constexpr int NWARPS = 4;
constexpr int PER_WARP = TS / NWARPS;

template <typename T> __device__ __forceinline__ float ld32(T x);
template <> __device__ __forceinline__ float ld32<float>(float x) { return x; }
template <> __device__ __forceinline__ float ld32<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T st32(float x);
template <> __device__ __forceinline__ float st32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 st32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

// delta[b, h, a] = <dO_a, O_a>: one warp per row
template <typename T, int D>
__global__ void __launch_bounds__(128) attn_bwd_delta_kernel(BwdParams prm) {
    const int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    const int64_t total = (int64_t)prm.B * prm.H * prm.Nq;
    if (row >= total) return;
    const int a = (int)(row % prm.Nq);
    const int h = (int)((row / prm.Nq) % prm.H), b = (int)(row / ((int64_t)prm.Nq * prm.H));
    const T *o = (const T *)prm.o.ptr + b * prm.o.stride_b + h * prm.o.stride_h + (int64_t)a * prm.o.stride_n;
    const T *g = (const T *)prm.dout.ptr + b * prm.dout.stride_b + h * prm.dout.stride_h + (int64_t)a * prm.dout.stride_n;
    float acc = 0.f;
    for (int c = lane; c < D; c += 32) acc = fmaf(ld32(o[c]), ld32(g[c]), acc);
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if (lane == 0) {
        if (prm.delta) prm.delta[row] = acc;
        if (prm.ld) prm.ld[row] = make_float2(prm.lse[row] * 1.4426950408889634f, acc);   // what the CTA-pair dQ pass consumes
        if (prm.aug) {
            // the 16 extra K columns of the CTA-pair dK/dV pass: v = h + l in bf16 (16 mantissa bits), stored halved in BOTH
            // 16-byte halves of the row (the constant A operand has ones at the same four positions): sum = v
            const float lse = prm.lse[row];
            const float v[2] = {lse == -CUDART_INF_F ? 0.f : -lse / prm.scale, -acc};   // rows without keys are never unmasked
            for (int i = 0; i < 2; ++i) {
                const __nv_bfloat16 h = __float2bfloat16_rn(v[i]);
                const __nv_bfloat16 l = __float2bfloat16_rn(v[i] - __bfloat162float(h));
                const __nv_bfloat16 h2 = __float2bfloat16_rn(0.5f * __bfloat162float(h)), l2 = __float2bfloat16_rn(0.5f * __bfloat162float(l));
                const uint32_t w = (uint32_t)__bfloat16_as_ushort(h2) | ((uint32_t)__bfloat16_as_ushort(l2) << 16);
                uint4 *dst = prm.aug + ((int64_t)i * total + row) * 2;
                dst[0] = make_uint4(w, 0u, 0u, 0u);
                dst[1] = make_uint4(w, 0u, 0u, 0u);
            }
        }
    }
}

// KEYS = false: stationary = query rows (Q, dO, lse, delta), streamed = keys (K, V); writes dQ.
// KEYS = true:  stationary = keys (K, V), streamed = query rows (Q, dO, lse, delta); writes dK, dV.
template <typename T, int D, bool KEYS>
__global__ void __launch_bounds__(NWARPS * 32) attn_bwd_simt_kernel(BwdParams prm) {
    constexpr int DP = D + 1;
    constexpr int DL = D / 32;
    extern __shared__ float smem[];
    float *sA = smem;               // stationary [TS][D]: Q (dQ pass) or K (dK/dV pass)
    float *sB = sA + TS * D;        // stationary [TS][D]: dO or V
    float *sC = sB + TS * D;        // streamed  [TM][DP]: K or Q
    float *sE = sC + TM * DP;       // streamed  [TM][DP]: V or dO
    float *sLse = sE + TM * DP;     // [max(TS, TM)] lse of the query rows (stationary or streamed)
    float *sDel = sLse + TM;        // delta likewise

    const aj_task task = (KEYS ? prm.k_tasks : prm.q_tasks)[blockIdx.x];
    const int32_t *rb = KEYS ? prm.k_rb : prm.q_kb, *re = KEYS ? prm.k_re : prm.q_ke;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const T *q = (const T *)prm.q.ptr + task.b * prm.q.stride_b + task.h * prm.q.stride_h;
    const T *k = (const T *)prm.k.ptr + task.b * prm.k.stride_b + task.h * prm.k.stride_h;
    const T *v = (const T *)prm.v.ptr + task.b * prm.v.stride_b + task.h * prm.v.stride_h;
    const T *g = (const T *)prm.dout.ptr + task.b * prm.dout.stride_b + task.h * prm.dout.stride_h;
    const float *lse = prm.lse + ((int64_t)task.b * prm.H + task.h) * prm.Nq;
    const float *del = prm.delta + ((int64_t)task.b * prm.H + task.h) * prm.Nq;
    const T *statA = KEYS ? k : q, *statB = KEYS ? v : g, *strC = KEYS ? q : k, *strE = KEYS ? g : v;
    const int64_t strideA = KEYS ? prm.k.stride_n : prm.q.stride_n, strideB = KEYS ? prm.v.stride_n : prm.dout.stride_n;
    const int64_t strideC = KEYS ? prm.q.stride_n : prm.k.stride_n, strideE = KEYS ? prm.dout.stride_n : prm.v.stride_n;

    for (int i = threadIdx.x; i < TS * D; i += blockDim.x) {
        const int r = i / D, c = i % D;
        const bool ok = r < task.q_rows;
        sA[i] = ok ? ld32(statA[(int64_t)(task.q_begin + r) * strideA + c]) : 0.f;
        sB[i] = ok ? ld32(statB[(int64_t)(task.q_begin + r) * strideB + c]) : 0.f;
    }
    if (!KEYS && threadIdx.x < TS) {
        const bool ok = threadIdx.x < task.q_rows;
        sLse[threadIdx.x] = ok ? lse[task.q_begin + threadIdx.x] : -CUDART_INF_F;
        sDel[threadIdx.x] = ok ? del[task.q_begin + threadIdx.x] : 0.f;
    }

    float acc1[PER_WARP][DL], acc2[PER_WARP][DL];   // dQ (acc1) | dK (acc1), dV (acc2)
#pragma unroll
    for (int i = 0; i < PER_WARP; ++i)
#pragma unroll
        for (int j = 0; j < DL; ++j) { acc1[i][j] = 0.f; acc2[i][j] = 0.f; }

    for (int ri = 0; ri < task.range_count; ++ri) {
        const int m0 = rb[task.range_begin + ri], m1 = re[task.range_begin + ri];
        for (int mt = m0; mt < m1; mt += TM) {
            __syncthreads();
            for (int i = threadIdx.x; i < TM * D; i += blockDim.x) {
                const int r = i / D, c = i % D;
                const bool ok = mt + r < m1;
                const int64_t row = mt + r;
                sC[r * DP + c] = ok ? ld32(strC[row * strideC + c]) : 0.f;
                sE[r * DP + c] = ok ? ld32(strE[row * strideE + c]) : 0.f;
            }
            if (KEYS && threadIdx.x < TM) {
                const bool ok = mt + threadIdx.x < m1;
                sLse[threadIdx.x] = ok ? lse[mt + threadIdx.x] : -CUDART_INF_F;
                sDel[threadIdx.x] = ok ? del[mt + threadIdx.x] : 0.f;
            }
            __syncthreads();
            const bool valid = mt + lane < m1;
#pragma unroll
            for (int i = 0; i < PER_WARP; ++i) {
                const int r = warp * PER_WARP + i;
                // the pair (stationary r, streamed lane): s = <q, k>, dP = <dO, v> whichever side is stationary
                const float *a = sA + r * D, *b = sB + r * D, *c = sC + lane * DP, *e = sE + lane * DP;
                float s = 0.f, dp = 0.f;
#pragma unroll 8
                for (int x = 0; x < D; ++x) {
                    s = fmaf(a[x], c[x], s);
                    dp = fmaf(b[x], e[x], dp);
                }
                const float l = KEYS ? sLse[lane] : sLse[r], dl = KEYS ? sDel[lane] : sDel[r];
                const float p = (valid && l > -CUDART_INF_F) ? expf(s * prm.scale - l) : 0.f;   // p_ab from the forward's lse
                const float ds = p * (dp - dl);                                                  // softmax Jacobian
                for (int x = 0; x < TM; ++x) {
                    const float dsx = __shfl_sync(0xffffffffu, ds, x);
                    const float px = __shfl_sync(0xffffffffu, p, x);
#pragma unroll
                    for (int j = 0; j < DL; ++j) {
                        acc1[i][j] = fmaf(dsx, sC[x * DP + lane + 32 * j], acc1[i][j]);          // dQ += dS k | dK += dS q
                        if (KEYS) acc2[i][j] = fmaf(px, sE[x * DP + lane + 32 * j], acc2[i][j]); // dV += p dO
                    }
                }
            }
        }
    }

    T *out1 = KEYS ? (T *)prm.dk.ptr + task.b * prm.dk.stride_b + task.h * prm.dk.stride_h
                   : (T *)prm.dq.ptr + task.b * prm.dq.stride_b + task.h * prm.dq.stride_h;
    T *out2 = KEYS ? (T *)prm.dv.ptr + task.b * prm.dv.stride_b + task.h * prm.dv.stride_h : nullptr;
    const int64_t so1 = KEYS ? prm.dk.stride_n : prm.dq.stride_n, so2 = prm.dv.stride_n;
#pragma unroll
    for (int i = 0; i < PER_WARP; ++i) {
        const int r = warp * PER_WARP + i;
        if (r >= task.q_rows) continue;
        const int64_t row = task.q_begin + r;
#pragma unroll
        for (int j = 0; j < DL; ++j) {
            out1[row * so1 + lane + 32 * j] = st32<T>(acc1[i][j] * prm.scale);
            if (KEYS) out2[row * so2 + lane + 32 * j] = st32<T>(acc2[i][j]);
        }
    }
}

template <typename T, int D>
cudaError_t launch_t(const BwdParams &prm, int num_q_tasks, int num_k_tasks, cudaStream_t stream) {
    const size_t smem = sizeof(float) * (2 * TS * D + 2 * TM * (D + 1) + 2 * TM);
    cudaError_t e = cudaFuncSetAttribute(attn_bwd_simt_kernel<T, D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(attn_bwd_simt_kernel<T, D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t rows = (int64_t)prm.B * prm.H * prm.Nq;
    attn_bwd_delta_kernel<T, D><<<(unsigned)((rows + 3) / 4), 128, 0, stream>>>(prm);
    if (num_q_tasks) attn_bwd_simt_kernel<T, D, false><<<num_q_tasks, NWARPS * 32, smem, stream>>>(prm);
    if (num_k_tasks) attn_bwd_simt_kernel<T, D, true><<<num_k_tasks, NWARPS * 32, smem, stream>>>(prm);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_bwd_delta(const BwdParams &prm, int dtype, int d, cudaStream_t stream) {
    const int64_t rows = (int64_t)prm.B * prm.H * prm.Nq;
    const unsigned grid = (unsigned)((rows + 3) / 4);
    if (dtype == AJ_BF16 && d == 128) attn_bwd_delta_kernel<__nv_bfloat16, 128><<<grid, 128, 0, stream>>>(prm);
    else if (dtype == AJ_BF16 && d == 64) attn_bwd_delta_kernel<__nv_bfloat16, 64><<<grid, 128, 0, stream>>>(prm);
    else if (dtype == AJ_FP32 && d == 128) attn_bwd_delta_kernel<float, 128><<<grid, 128, 0, stream>>>(prm);
    else if (dtype == AJ_FP32 && d == 64) attn_bwd_delta_kernel<float, 64><<<grid, 128, 0, stream>>>(prm);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

cudaError_t launch_bwd_simt(const BwdParams &prm, int dtype, int d, int num_q_tasks, int num_k_tasks, cudaStream_t stream) {
    if (dtype == AJ_FP32 && d == 64) return launch_t<float, 64>(prm, num_q_tasks, num_k_tasks, stream);
    if (dtype == AJ_FP32 && d == 128) return launch_t<float, 128>(prm, num_q_tasks, num_k_tasks, stream);
    if (dtype == AJ_BF16 && d == 64) return launch_t<__nv_bfloat16, 64>(prm, num_q_tasks, num_k_tasks, stream);
    if (dtype == AJ_BF16 && d == 128) return launch_t<__nv_bfloat16, 128>(prm, num_q_tasks, num_k_tasks, stream);
    return cudaErrorInvalidValue;
}

}  // namespace aj
