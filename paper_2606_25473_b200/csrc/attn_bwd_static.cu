// attn_bwd_static: the primal backward for callers that must not allocate (include/attn_jvp.h has the contract).
//
// Who this is for.  attn_bwd gets its schedules and its [B, H, Nq] `delta` workspace from cudaMalloc on a plan's first call,
// and a plan itself is device memory.  Two kinds of host program cannot live with that:
//   * a process whose own pool took the GPU's memory at start-up (a training or serving framework with a caching allocator
//     that reserves the whole card): a cudaMalloc made behind its back by a library either fails with out-of-memory or takes
//     memory the pool has already promised to someone else;
//   * a loop with a latency budget and other streams in flight: cudaMalloc and cudaFree may serialise against all work on
//     the device, so one allocation inside a step stalls every stream, not just the caller's.
// For them this file computes the same dQ, dK, dV with no plan and no allocation of any kind.  The only memory the kernels
// touch besides the caller's tensors is `g_delta_scratch` below: a fixed array that is part of the library's device image.
//
// What it computes (PAPER.md:247, Eq. 19: the student's gradient flows through the primal path; :945: the forward returns
// L for it).  With p_ab = exp(s <q_a, k_b> - lse_a) over the unmasked pairs:
//     delta_a = <dO_a, O_a>,  dS_ab = p_ab (<dO_a, v_b> - delta_a),
//     dQ_a = s sum_b dS_ab k_b,  dK_b = s sum_a dS_ab q_a,  dV_b = sum_a p_ab dO_a.
// The kernels are a variant of the plain-FMA backward of kernel_simt_bwd.cu (same tiles, same fp32 arithmetic) that needs no
// schedule in device memory: a CTA derives its tile from blockIdx and decides pair by pair, from four integers, whether the
// mask admits it (PAPER.md:175-180 teacher forcing, :155 block-causal, :886 dense), skipping streamed tiles that hold no
// admitted pair.  It is a correctness-grade path (a few TFLOP/s), not the tcgen05 one.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include <cmath>
#include <mutex>
#include <string>

#include "internal.hpp"

// The scratch: delta_a for every query row of one call.  AJ_STATIC_SCRATCH_MAX_ROWS floats = 4 MiB, resident on every GPU
// that loads the library until the process exits.  In HOST code this name is only a handle for cudaGetSymbolAddress, never a
// device address; the launchers below pass the address they looked up.
static __device__ __align__(256) float g_delta_scratch[AJ_STATIC_SCRATCH_MAX_ROWS];

namespace {

using aj::fail;

constexpr int TS = 16;   // stationary rows per CTA (query rows for dQ, keys for dK / dV)
constexpr int TM = 32;   // streamed rows per tile: one per lane
constexpr int NWARPS = 4;
constexpr int PER_WARP = TS / NWARPS;

// The structured masks as integers (tokens): a half holds `half` tokens, its block 0 the first `first` of them, every later
// block `chunk`.  kind is an aj_mask_kind (never RANGES).
struct MaskRule {
    int32_t kind, half, first, chunk;
};

__device__ __forceinline__ int block_of(const MaskRule &m, int t) { return t < m.first ? 0 : 1 + (t - m.first) / m.chunk; }

// Does query row a see key b?
__device__ __forceinline__ bool admits(const MaskRule &m, int a, int b) {
    if (m.kind == AJ_MASK_FULL) return true;
    if (m.kind == AJ_MASK_BLOCK_CAUSAL) return block_of(m, b) <= block_of(m, a);
    // teacher forcing over [clean | noisy]
    if (a < m.half) return b < m.half && block_of(m, b) <= block_of(m, a);
    const int ia = block_of(m, a - m.half);
    return b < m.half ? block_of(m, b) < ia : block_of(m, b - m.half) == ia;
}

struct StaticParams {
    aj_tensor q, k, v, o, dout, dq, dk, dv;
    const float *lse;   // [B, H, Nq]
    float *delta;       // the scratch, by device address
    MaskRule mask;
    int32_t B, H, Nq, Nk;
    float scale;
};

template <typename T> __device__ __forceinline__ float ld32(T x);
template <> __device__ __forceinline__ float ld32<float>(float x) { return x; }
template <> __device__ __forceinline__ float ld32<__nv_bfloat16>(__nv_bfloat16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T st32(float x);
template <> __device__ __forceinline__ float st32<float>(float x) { return x; }
template <> __device__ __forceinline__ __nv_bfloat16 st32<__nv_bfloat16>(float x) { return __float2bfloat16_rn(x); }

// delta[row] = <dO_row, O_row>, one warp per row.  Every entry a later kernel of the same call reads is written here first,
// so nothing in the scratch has to start at zero and whatever an earlier call left behind is never seen.
template <typename T, int D>
__global__ void __launch_bounds__(128) static_delta_kernel(StaticParams prm) {
    const int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (row >= (int64_t)prm.B * prm.H * prm.Nq) return;
    const int a = (int)(row % prm.Nq);
    const int h = (int)((row / prm.Nq) % prm.H), b = (int)(row / ((int64_t)prm.Nq * prm.H));
    const T *o = (const T *)prm.o.ptr + b * prm.o.stride_b + h * prm.o.stride_h + (int64_t)a * prm.o.stride_n;
    const T *g = (const T *)prm.dout.ptr + b * prm.dout.stride_b + h * prm.dout.stride_h + (int64_t)a * prm.dout.stride_n;
    float acc = 0.f;
    for (int c = lane; c < D; c += 32) acc = fmaf(ld32(o[c]), ld32(g[c]), acc);
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if (lane == 0) prm.delta[row] = acc;
}

// KEYS = false: TS query rows stay (Q, dO, lse, delta), keys stream (K, V); writes dQ.
// KEYS = true:  TS keys stay (K, V), query rows stream (Q, dO, lse, delta); writes dK, dV.
// blockIdx.x = (b * H + h) * tiles + tile.
template <typename T, int D, bool KEYS>
__global__ void __launch_bounds__(NWARPS * 32) static_bwd_kernel(StaticParams prm) {
    constexpr int DP = D + 1;
    constexpr int DL = D / 32;
    extern __shared__ float smem[];
    float *sA = smem;               // stationary [TS][D]: Q or K
    float *sB = sA + TS * D;        // stationary [TS][D]: dO or V
    float *sC = sB + TS * D;        // streamed  [TM][DP]: K or Q
    float *sE = sC + TM * DP;       // streamed  [TM][DP]: V or dO
    float *sLse = sE + TM * DP;     // [TM] lse of the query rows (stationary or streamed)
    float *sDel = sLse + TM;        // delta likewise

    const int n_stat = KEYS ? prm.Nk : prm.Nq, n_str = KEYS ? prm.Nq : prm.Nk;
    const int tiles = (n_stat + TS - 1) / TS;
    const int tile = blockIdx.x % tiles, head = blockIdx.x / tiles;
    const int hb = head / prm.H, hh = head % prm.H;
    const int s0 = tile * TS, s_rows = min(TS, n_stat - s0);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const T *q = (const T *)prm.q.ptr + hb * prm.q.stride_b + hh * prm.q.stride_h;
    const T *k = (const T *)prm.k.ptr + hb * prm.k.stride_b + hh * prm.k.stride_h;
    const T *v = (const T *)prm.v.ptr + hb * prm.v.stride_b + hh * prm.v.stride_h;
    const T *g = (const T *)prm.dout.ptr + hb * prm.dout.stride_b + hh * prm.dout.stride_h;
    const float *lse = prm.lse + (int64_t)head * prm.Nq;
    const float *del = prm.delta + (int64_t)head * prm.Nq;
    const T *statA = KEYS ? k : q, *statB = KEYS ? v : g, *strC = KEYS ? q : k, *strE = KEYS ? g : v;
    const int64_t strideA = KEYS ? prm.k.stride_n : prm.q.stride_n, strideB = KEYS ? prm.v.stride_n : prm.dout.stride_n;
    const int64_t strideC = KEYS ? prm.q.stride_n : prm.k.stride_n, strideE = KEYS ? prm.dout.stride_n : prm.v.stride_n;

    for (int i = threadIdx.x; i < TS * D; i += blockDim.x) {
        const int r = i / D, c = i % D;
        const bool ok = r < s_rows;
        sA[i] = ok ? ld32(statA[(int64_t)(s0 + r) * strideA + c]) : 0.f;
        sB[i] = ok ? ld32(statB[(int64_t)(s0 + r) * strideB + c]) : 0.f;
    }
    if (!KEYS && threadIdx.x < TS) {
        const bool ok = threadIdx.x < s_rows;
        sLse[threadIdx.x] = ok ? lse[s0 + threadIdx.x] : -CUDART_INF_F;
        sDel[threadIdx.x] = ok ? del[s0 + threadIdx.x] : 0.f;
    }

    float acc1[PER_WARP][DL], acc2[PER_WARP][DL];   // dQ (acc1) | dK (acc1), dV (acc2)
#pragma unroll
    for (int i = 0; i < PER_WARP; ++i)
#pragma unroll
        for (int j = 0; j < DL; ++j) { acc1[i][j] = 0.f; acc2[i][j] = 0.f; }

    // pair (stationary r, streamed x) of the current tile as (query row, key)
    auto seen = [&](int r, int x) {
        const int s = s0 + r;
        if (r >= s_rows || x >= n_str) return false;
        return KEYS ? admits(prm.mask, x, s) : admits(prm.mask, s, x);
    };

    for (int mt = 0; mt < n_str; mt += TM) {
        // does the mask admit any of the tile's TS x TM pairs?  Thread t looks at stationary row t % TS and four streamed rows.
        bool any = false;
        if (prm.mask.kind == AJ_MASK_FULL) {
            any = true;
        } else {
            const int r = threadIdx.x % TS, x0 = mt + (threadIdx.x / TS) * 4;
#pragma unroll
            for (int x = 0; x < 4; ++x) any = any || seen(r, x0 + x);
        }
        if (!__syncthreads_or(any)) continue;     // also the barrier that protects sC / sE of the previous tile
        for (int i = threadIdx.x; i < TM * D; i += blockDim.x) {
            const int r = i / D, c = i % D;
            const bool ok = mt + r < n_str;
            const int64_t row = mt + r;
            sC[r * DP + c] = ok ? ld32(strC[row * strideC + c]) : 0.f;
            sE[r * DP + c] = ok ? ld32(strE[row * strideE + c]) : 0.f;
        }
        if (KEYS && threadIdx.x < TM) {
            const bool ok = mt + threadIdx.x < n_str;
            sLse[threadIdx.x] = ok ? lse[mt + threadIdx.x] : -CUDART_INF_F;
            sDel[threadIdx.x] = ok ? del[mt + threadIdx.x] : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < PER_WARP; ++i) {
            const int r = warp * PER_WARP + i;
            const float *a = sA + r * D, *b = sB + r * D, *c = sC + lane * DP, *e = sE + lane * DP;
            float s = 0.f, dp = 0.f;
#pragma unroll 8
            for (int x = 0; x < D; ++x) {
                s = fmaf(a[x], c[x], s);       // <q, k>
                dp = fmaf(b[x], e[x], dp);     // <dO, v>
            }
            const float l = KEYS ? sLse[lane] : sLse[r], dl = KEYS ? sDel[lane] : sDel[r];
            const float p = (seen(r, mt + lane) && l > -CUDART_INF_F) ? expf(s * prm.scale - l) : 0.f;
            const float ds = p * (dp - dl);
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

    T *out1 = KEYS ? (T *)prm.dk.ptr + hb * prm.dk.stride_b + hh * prm.dk.stride_h
                   : (T *)prm.dq.ptr + hb * prm.dq.stride_b + hh * prm.dq.stride_h;
    T *out2 = KEYS ? (T *)prm.dv.ptr + hb * prm.dv.stride_b + hh * prm.dv.stride_h : nullptr;
    const int64_t so1 = KEYS ? prm.dk.stride_n : prm.dq.stride_n, so2 = prm.dv.stride_n;
#pragma unroll
    for (int i = 0; i < PER_WARP; ++i) {
        const int r = warp * PER_WARP + i;
        if (r >= s_rows) continue;
        const int64_t row = s0 + r;
#pragma unroll
        for (int j = 0; j < DL; ++j) {
            out1[row * so1 + lane + 32 * j] = st32<T>(acc1[i][j] * prm.scale);
            if (KEYS) out2[row * so2 + lane + 32 * j] = st32<T>(acc2[i][j]);
        }
    }
}

constexpr size_t smem_bytes(int d) { return sizeof(float) * (size_t)(2 * TS * d + 2 * TM * (d + 1) + 2 * TM); }

// Per-device set-up, done by the first call that runs with that device current: the scratch's address ON THAT DEVICE
// (cudaGetSymbolAddress answers for the current device; the array exists once per GPU) and the shared-memory opt-in of the
// kernels that need more than 48 KB.  Neither allocates; the first may make the runtime load the library's device image.
struct DeviceSetup {
    float *scratch = nullptr;
    bool ready = false;
};
constexpr int MAX_DEVICES = 64;
DeviceSetup g_setup[MAX_DEVICES];
std::mutex g_setup_mu;

template <typename T, int D>
cudaError_t opt_in_smem() {
    cudaError_t e = cudaFuncSetAttribute(static_bwd_kernel<T, D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(D));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(static_bwd_kernel<T, D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(D));
    return e;
}

aj_status device_scratch(float **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(AJ_ERR_CUDA, std::string("attn_bwd_static: cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(AJ_ERR_UNSUPPORTED, "attn_bwd_static: device ordinals above 63 are not supported");
    std::lock_guard<std::mutex> lock(g_setup_mu);
    DeviceSetup &s = g_setup[dev];
    if (!s.ready) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_delta_scratch);
        if (e == cudaSuccess) e = opt_in_smem<float, 64>();
        if (e == cudaSuccess) e = opt_in_smem<float, 128>();
        if (e == cudaSuccess) e = opt_in_smem<__nv_bfloat16, 64>();
        if (e == cudaSuccess) e = opt_in_smem<__nv_bfloat16, 128>();
        if (e != cudaSuccess) return fail(AJ_ERR_CUDA, std::string("attn_bwd_static: set-up on device ") + std::to_string(dev) + ": " + cudaGetErrorString(e));
        if (!p) return fail(AJ_ERR_CUDA, "attn_bwd_static: cudaGetSymbolAddress returned a null address");
        s.scratch = (float *)p;
        s.ready = true;
    }
    *out = s.scratch;
    return AJ_OK;
}

template <typename T, int D>
cudaError_t launch_t(const StaticParams &prm, cudaStream_t stream) {
    const int64_t rows = (int64_t)prm.B * prm.H * prm.Nq;
    const int64_t heads = (int64_t)prm.B * prm.H;
    const unsigned q_tiles = (unsigned)(heads * ((prm.Nq + TS - 1) / TS)), k_tiles = (unsigned)(heads * ((prm.Nk + TS - 1) / TS));
    static_delta_kernel<T, D><<<(unsigned)((rows + 3) / 4), 128, 0, stream>>>(prm);
    static_bwd_kernel<T, D, false><<<q_tiles, NWARPS * 32, smem_bytes(D), stream>>>(prm);
    static_bwd_kernel<T, D, true><<<k_tiles, NWARPS * 32, smem_bytes(D), stream>>>(prm);
    return cudaGetLastError();
}

// the same rules as the planned calls: 16-byte aligned pointers, strides in multiples of 8 elements, stride_n >= d; inputs may be
// broadcast over heads / batches with a zero stride, outputs may not
aj_status check_view(const aj_tensor *t, const char *name, const aj_problem &p, bool output) {
    if (!t || !t->ptr) return fail(AJ_ERR_INVALID_ARG, std::string("attn_bwd_static: ") + name + " is NULL");
    if ((uintptr_t)t->ptr % 16 != 0) return fail(AJ_ERR_INVALID_ARG, std::string("attn_bwd_static: ") + name + ": pointer must be 16-byte aligned");
    if (t->stride_n < p.d || t->stride_n % 8 || t->stride_h % 8 || t->stride_b % 8 || t->stride_h < 0 || t->stride_b < 0)
        return fail(AJ_ERR_INVALID_ARG, std::string("attn_bwd_static: ") + name + ": strides must be multiples of 8 elements with stride_n >= d");
    if (output && ((p.H > 1 && t->stride_h == 0) || (p.B > 1 && t->stride_b == 0)))
        return fail(AJ_ERR_INVALID_ARG, std::string("attn_bwd_static: ") + name + ": an output tensor must not alias heads or batches (zero stride)");
    return AJ_OK;
}

aj_status mask_rule(const aj_problem &p, const aj_mask_desc &m, MaskRule &out) {
    out = MaskRule{m.kind, 0, 0, 1};
    if (m.kind == AJ_MASK_FULL) return AJ_OK;
    if (m.kind == AJ_MASK_RANGES)
        return fail(AJ_ERR_UNSUPPORTED, "attn_bwd_static: AJ_MASK_RANGES needs its range lists in device memory, which this call does not own; use attn_bwd");
    if (m.kind != AJ_MASK_BLOCK_CAUSAL && m.kind != AJ_MASK_TEACHER_FORCING) return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: unknown mask kind");
    if (m.frame_len <= 0 || m.num_frames <= 0 || m.chunk_frames <= 0 || m.first_chunk_frames < 0)
        return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: mask: frame_len, num_frames, chunk_frames must be > 0");
    const int64_t first = m.first_chunk_frames > 0 ? m.first_chunk_frames : m.chunk_frames;
    if (first > m.num_frames || (m.num_frames - first) % m.chunk_frames != 0)
        return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: mask: num_frames is not first_chunk_frames + k * chunk_frames");
    const int64_t half = (int64_t)m.num_frames * m.frame_len, n = m.kind == AJ_MASK_TEACHER_FORCING ? 2 * half : half;
    if (p.Nq != n || p.Nk != n)
        return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: Nq and Nk must equal num_frames * frame_len (twice that for teacher forcing)");
    out.half = (int32_t)half;
    out.first = (int32_t)(first * m.frame_len);
    out.chunk = (int32_t)((int64_t)m.chunk_frames * m.frame_len);
    return AJ_OK;
}

}  // namespace

extern "C" aj_status attn_bwd_static(const aj_problem *problem, const aj_mask_desc *mask, const aj_tensor *q, const aj_tensor *k,
                                     const aj_tensor *v, const aj_tensor *o, const float *lse, const aj_tensor *dout,
                                     const aj_tensor *dq, const aj_tensor *dk, const aj_tensor *dv, void *cuda_stream) {
    if (aj_status st = aj::check_problem(problem)) return st;
    if (!mask) return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: mask is NULL");
    aj_problem pr = *problem;
    if (pr.d != 64 && pr.d != 128) return fail(AJ_ERR_UNSUPPORTED, "attn_bwd_static: d must be 64 or 128");
    if (pr.scale == 0.0f) pr.scale = 1.0f / std::sqrt((float)pr.d);
    StaticParams prm;
    if (aj_status st = mask_rule(pr, *mask, prm.mask)) return st;
    // the one size limit: a call's query rows must fit the fixed scratch
    const int64_t rows = (int64_t)pr.B * pr.H * pr.Nq;
    if (rows > (int64_t)AJ_STATIC_SCRATCH_MAX_ROWS)
        return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: B * H * Nq = " + std::to_string(rows) + " query rows exceed the fixed scratch of AJ_STATIC_SCRATCH_MAX_ROWS = " +
                                            std::to_string((int64_t)AJ_STATIC_SCRATCH_MAX_ROWS) + " rows; split the call over heads or use attn_bwd");
    if ((int64_t)pr.B * pr.H * (((int64_t)pr.Nk + TS - 1) / TS) > 0x7fffffffLL)
        return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: B * H * Nk is too large for one launch");
    const aj_tensor *ts[8] = {q, k, v, o, dout, dq, dk, dv};
    const char *names[8] = {"q", "k", "v", "o", "dout", "dq", "dk", "dv"};
    for (int i = 0; i < 8; ++i)
        if (aj_status st = check_view(ts[i], names[i], pr, i >= 5)) return st;
    if (!lse || (uintptr_t)lse % 4 != 0) return fail(AJ_ERR_INVALID_ARG, "attn_bwd_static: lse is NULL or misaligned");
    if (aj_status st = device_scratch(&prm.delta)) return st;
    prm.q = *q; prm.k = *k; prm.v = *v; prm.o = *o; prm.dout = *dout; prm.dq = *dq; prm.dk = *dk; prm.dv = *dv;
    prm.lse = lse;
    prm.B = pr.B; prm.H = pr.H; prm.Nq = pr.Nq; prm.Nk = pr.Nk; prm.scale = pr.scale;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (pr.dtype == AJ_FP32 && pr.d == 64) e = launch_t<float, 64>(prm, stream);
    else if (pr.dtype == AJ_FP32) e = launch_t<float, 128>(prm, stream);
    else if (pr.d == 64) e = launch_t<__nv_bfloat16, 64>(prm, stream);
    else e = launch_t<__nv_bfloat16, 128>(prm, stream);
    if (e != cudaSuccess) return fail(AJ_ERR_CUDA, std::string("attn_bwd_static: kernel launch: ") + cudaGetErrorString(e));
    return AJ_OK;
}
