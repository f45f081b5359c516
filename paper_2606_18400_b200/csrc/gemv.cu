// S6 cloak_gemv: decode GEMV (batch 1..16) that reads W through the block table.
//
// Definition (north_star (c) "gather-fused GEMV (warp-level split-K reductions,
// bandwidth-bound)"; "LLM inference is bandwidth-bound"):
//     Y[m, n] = sum_k X[m, k] * W[n, k],  W row-major [N, K] at arena offset w_offset,
//     byte x of the arena lives at  pool + (T[x >> log2 b] << log2 b) + (x & (b - 1)).
// Weight bytes are read exactly once (N*K*e algorithmic bytes); HBM-bound.
//
// bf16 kernel.  One CTA = 16 output rows, 4 warps splitting K (split-K, reduced through shared memory in a
// fixed order -> deterministic, and bit-identical between a cloaked and an identity-table pool).  Each lane
// (g = lane/4, t = lane%4) loads 16-byte vectors W[g][k0+8t .. +8) and W[g+8][...], i.e. every load
// instruction of a warp covers 8 rows x 64 contiguous bytes; two of them (k0, k0+32) consume whole 128-byte
// lines.  The 8 bf16 of a vector feed two mma.sync.m16n8k16 (bf16 in, fp32 accumulate) as the A operand with
// the batch as the N=8 operand: because a contraction may visit k in any order, lane t's vector elements
// (8t+0..3 / 8t+4..7) are *declared* to be the MMA's k-slots (2t,2t+1,2t+8,2t+9); the X fragment is loaded
// with the same rule (one 16-byte load of X[g][k0+8t .. +8)), so no shuffle or shared-memory transpose is
// needed and the batch costs no extra weight traffic.  Tensor-pipe demand is ~0.1 PFLOP/s at batch 16:
// the kernel stays on the HBM roofline where plain FMAs (52 TFMA/s needed, 37 available) could not.
//
// fp32 kernel (cfg0, correctness path): one warp per row, 16-byte loads, fp32 FMA, shuffle reduction.
#include <cuda_bf16.h>
#include "common.cuh"

namespace cloak {

struct GemvArgs {
    const char* pool;
    const uint32_t* T;
    uint32_t log2b;
    uint64_t w_offset;
    uint32_t N, K;
    const void* x;
    void* y;
    uint32_t batch;
    uint32_t zero;      // always 0; see the scheduling fence in gemv_bf16_kernel
};

__device__ __forceinline__ const char* xlate(const GemvArgs& a, uint64_t off) {
    const uint32_t slot = __ldg(a.T + (off >> a.log2b));
    return a.pool + ((uint64_t)slot << a.log2b) + (off & ((1ull << a.log2b) - 1));
}

__device__ __forceinline__ uint4 ld_w(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ void mma_bf16_16816(float c[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

constexpr int GV_WARPS = 4;
constexpr int GV_ROWS = 16;
constexpr int GV_KSTEP = 64;                          // k elements per warp step: 2 vectors per row per lane
constexpr int GV_STEPS = 4;                           // k-steps per warp: all issued before the first MMA
constexpr int GV_KCTA = GV_WARPS * GV_STEPS * GV_KSTEP;   // 1024 k elements per CTA
constexpr uint32_t GV_MAX_TILES = (uint32_t)(WS_COUNTER_BYTES / 4);          // row tiles per launch the split-K counters cover

// One CTA = 16 rows x 1024 k, one shot: every lane issues its 16 weight loads (8 KiB per warp, 32 KiB per
// CTA) before the first MMA, so the bytes in flight per SM are occupancy x 32 KiB with no loop-carried
// latency and a tail of one short CTA lifetime.  K is split over S = ceil(K/1024) CTAs (blockIdx = tile*S+s).
// S > 1: every CTA stores its fp32 partial, and the last CTA to arrive at the tile's counter sums the S
// partials in s order (fixed order -> deterministic, bit-identical between cloaked and identity pools).
// FULL: K is a multiple of 1024, so no k-step needs a bounds check.
template <int NT, bool FULL>   // NT = number of 8-wide batch tiles (1: batch <= 8, 2: batch <= 16)
__global__ void __launch_bounds__(GV_WARPS * 32) gemv_bf16_kernel(GemvArgs a, uint32_t S, float* __restrict__ part,
                                                                  uint32_t* __restrict__ counters) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const uint32_t tile = blockIdx.x / S, split = blockIdx.x - tile * S;
    const uint32_t n0 = tile * GV_ROWS;
    const uint32_t kbase = split * GV_KCTA + warp * (GV_STEPS * GV_KSTEP);
    const uint64_t row_lo = a.w_offset + ((uint64_t)(n0 + g) * a.K + kbase + t * 8) * 2;
    const uint64_t row_hi = row_lo + (uint64_t)8 * a.K * 2;
    const uint16_t* X = static_cast<const uint16_t*>(a.x);
    const bool xv0 = (uint32_t)g < a.batch, xv1 = (uint32_t)(g + 8) < a.batch;
    const uint16_t* x0 = X + (size_t)g * a.K + kbase + t * 8;
    const uint16_t* x1 = X + (size_t)(g + 8) * a.K + kbase + t * 8;

    // All table lookups first (independent L2 hits), then all 16 weight loads: nothing serialises.
    const char* pl[GV_STEPS];
    const char* ph[GV_STEPS];
#pragma unroll
    for (int u = 0; u < GV_STEPS; ++u) {
        const bool in = FULL || kbase + u * GV_KSTEP < a.K;
        pl[u] = in ? xlate(a, row_lo + (uint64_t)u * GV_KSTEP * 2) : nullptr;   // 128-byte line of row g
        ph[u] = in ? xlate(a, row_hi + (uint64_t)u * GV_KSTEP * 2) : nullptr;   // 128-byte line of row g+8
    }
    uint4 wl[GV_STEPS][2], wh[GV_STEPS][2];
#pragma unroll
    for (int u = 0; u < GV_STEPS; ++u) {
        if (FULL || pl[u]) {
            wl[u][0] = ld_w(pl[u]);
            wl[u][1] = ld_w(pl[u] + 64);
            wh[u][0] = ld_w(ph[u]);
            wh[u][1] = ld_w(ph[u] + 64);
        }
    }
    // The activations (L2-resident, shared by every CTA) are requested right behind the weights.
    uint4 xa[GV_STEPS][2], xb[GV_STEPS][2];
#pragma unroll
    for (int u = 0; u < GV_STEPS; ++u) {
        const uint4 z = make_uint4(0, 0, 0, 0);
        const bool in = FULL || kbase + u * GV_KSTEP < a.K;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            xa[u][h] = (xv0 && in) ? __ldg(reinterpret_cast<const uint4*>(x0 + u * GV_KSTEP + h * 32)) : z;
            if (NT == 2) xb[u][h] = (xv1 && in) ? __ldg(reinterpret_cast<const uint4*>(x1 + u * GV_KSTEP + h * 32)) : z;
        }
    }
    // Scheduling fence.  ptxas otherwise sinks the loads between the MMAs to save registers, which
    // serialises the memory latency.  The accumulators are seeded with (xor of one word of every weight
    // vector) & a.zero -- a.zero is 0 at run time but opaque to the compiler -- so the first MMA of each
    // chain depends on all 16 loads and every request is in flight before any of them is consumed.
    uint32_t dep = 0;
#pragma unroll
    for (int u = 0; u < GV_STEPS; ++u)
        if (FULL || pl[u]) dep ^= wl[u][0].x ^ wl[u][1].x ^ wh[u][0].x ^ wh[u][1].x;
    const float seed = __uint_as_float(dep & a.zero);
    float acc[NT][4];
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = seed;
#pragma unroll
    for (int u = 0; u < GV_STEPS; ++u) {
        if (FULL || kbase + u * GV_KSTEP < a.K) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                mma_bf16_16816(acc[0], wl[u][h].x, wh[u][h].x, wl[u][h].y, wh[u][h].y, xa[u][h].x, xa[u][h].y);
                mma_bf16_16816(acc[0], wl[u][h].z, wh[u][h].z, wl[u][h].w, wh[u][h].w, xa[u][h].z, xa[u][h].w);
                if (NT == 2) {
                    mma_bf16_16816(acc[1], wl[u][h].x, wh[u][h].x, wl[u][h].y, wh[u][h].y, xb[u][h].x, xb[u][h].y);
                    mma_bf16_16816(acc[1], wl[u][h].z, wh[u][h].z, wl[u][h].w, wh[u][h].w, xb[u][h].z, xb[u][h].w);
                }
            }
        }
    }

    // In-CTA split-K reduction across the 4 warps in fixed order.
    __shared__ float red[GV_WARPS][NT * 8][GV_ROWS + 1];      // [warp][batch m][row]
    __shared__ uint32_t is_last;
#pragma unroll
    for (int i = 0; i < NT; ++i) {
        red[warp][i * 8 + 2 * t][g] = acc[i][0];
        red[warp][i * 8 + 2 * t + 1][g] = acc[i][1];
        red[warp][i * 8 + 2 * t][g + 8] = acc[i][2];
        red[warp][i * 8 + 2 * t + 1][g + 8] = acc[i][3];
    }
    __syncthreads();
    __nv_bfloat16* Y = static_cast<__nv_bfloat16*>(a.y);
    const uint32_t nout = a.batch * GV_ROWS;
    if (S == 1) {
        for (uint32_t i = threadIdx.x; i < nout; i += blockDim.x) {
            const uint32_t m = i / GV_ROWS, r = i % GV_ROWS;
            float s = red[0][m][r];
#pragma unroll
            for (int w = 1; w < GV_WARPS; ++w) s += red[w][m][r];
            Y[(size_t)m * a.N + n0 + r] = __float2bfloat16_rn(s);
        }
        return;
    }
    // Cross-CTA split-K: partial[split][m][n], then the last arriver reduces in split order.
    for (uint32_t i = threadIdx.x; i < nout; i += blockDim.x) {
        const uint32_t m = i / GV_ROWS, r = i % GV_ROWS;
        float s = red[0][m][r];
#pragma unroll
        for (int w = 1; w < GV_WARPS; ++w) s += red[w][m][r];
        __stcg(part + ((size_t)split * a.batch + m) * a.N + n0 + r, s);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t old = atomicAdd(counters + tile, 1u);
        is_last = (old == S - 1);
        if (old == S - 1) counters[tile] = 0;          // self-reset for the next launch
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (uint32_t i = threadIdx.x; i < nout; i += blockDim.x) {
        const uint32_t m = i / GV_ROWS, r = i % GV_ROWS;
        float s = 0.f;
        for (uint32_t q = 0; q < S; ++q) s += __ldcg(part + ((size_t)q * a.batch + m) * a.N + n0 + r);
        Y[(size_t)m * a.N + n0 + r] = __float2bfloat16_rn(s);
    }
}

// fp32: one warp per output row; lanes stride K in float4; batch accumulators in registers.
template <int MB>
__global__ void __launch_bounds__(256) gemv_f32_kernel(GemvArgs a) {
    const int lane = threadIdx.x & 31;
    const uint32_t row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= a.N) return;
    const float* X = static_cast<const float*>(a.x);
    float acc[MB];
#pragma unroll
    for (int m = 0; m < MB; ++m) acc[m] = 0.f;
    const uint64_t row_off = a.w_offset + (uint64_t)row * a.K * 4;
    for (uint32_t k = lane * 4; k < a.K; k += 128) {
        const float4 w = *reinterpret_cast<const float4*>(xlate(a, row_off + (uint64_t)k * 4));
#pragma unroll
        for (int m = 0; m < MB; ++m) {
            if ((uint32_t)m < a.batch) {
                const float4 x = __ldg(reinterpret_cast<const float4*>(X + (size_t)m * a.K + k));
                acc[m] = fmaf(w.x, x.x, acc[m]);
                acc[m] = fmaf(w.y, x.y, acc[m]);
                acc[m] = fmaf(w.z, x.z, acc[m]);
                acc[m] = fmaf(w.w, x.w, acc[m]);
            }
        }
    }
    float* Y = static_cast<float*>(a.y);
#pragma unroll
    for (int m = 0; m < MB; ++m) {
        float s = acc[m];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0 && (uint32_t)m < a.batch) Y[(size_t)m * a.N + row] = s;
    }
}

cloak_status check_linear(const cloak_pool* pool, const cloak_tensor* w, const void* x, void* y, const char* who) {
    if (!pool || !w || !x || !y) return fail(CLOAK_ERR_INVALID, "%s: NULL argument", who);
    if (w->dt != CLOAK_F32 && w->dt != CLOAK_BF16) return fail(CLOAK_ERR_UNSUPPORTED, "%s: unknown dtype", who);
    if (w->N == 0 || w->K == 0) return fail(CLOAK_ERR_INVALID, "%s: empty tensor", who);
    if (w->w_offset % pool->block) return fail(CLOAK_ERR_ALIGN, "%s: w_offset is not a block multiple", who);
    const uint64_t bytes = (uint64_t)w->N * w->K * (w->dt == CLOAK_F32 ? 4 : 2);
    if (w->w_offset + bytes > (uint64_t)pool->nb * pool->block) return fail(CLOAK_ERR_INVALID, "%s: tensor exceeds the pool's arena", who);
    if (((uintptr_t)x | (uintptr_t)y) & 15) return fail(CLOAK_ERR_ALIGN, "%s: x / y not 16-byte aligned", who);
    return CLOAK_OK;
}

// Library-owned scratch of a pool: WS_COUNTER_BYTES of self-resetting split-K counters (zeroed when allocated) followed
// by fp32 partials.  Calls that use it on one pool must be stream-ordered with respect to each other.  Growth happens in
// the order of stream `s`: the new buffer is allocated and its counters zeroed on s, the old one is freed on s, so
// kernels already queued keep theirs; nothing synchronises.  Impossible while s is being captured into a graph (the
// buffer would belong to the graph): cloak_pool_reserve_workspace beforehand.
cloak_status pool_workspace(const cloak_pool* pool, size_t bytes, cudaStream_t s) {
    if (pool->ws_bytes >= bytes) return CLOAK_OK;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &cap) != cudaSuccess) cudaGetLastError();
    if (cap != cudaStreamCaptureStatusNone)
        return fail(CLOAK_ERR_INVALID, "this call needs %zu bytes of pool scratch (the pool has %zu) and the stream is being captured: "
                                       "call cloak_pool_reserve_workspace before the capture", bytes, pool->ws_bytes);
    const size_t want = bytes < WS_DEFAULT_BYTES ? WS_DEFAULT_BYTES : bytes;
    void* nw = nullptr;
    cloak_status st = async_alloc(&nw, want, s);
    if (st != CLOAK_OK) return st;
    CLOAK_CUDA(cudaMemsetAsync(nw, 0, WS_COUNTER_BYTES, s));
    if (pool->ws) CLOAK_CUDA(cudaFreeAsync(pool->ws, s));
    pool->ws = static_cast<char*>(nw);
    pool->ws_bytes = want;
    return CLOAK_OK;
}

static std::atomic<bool> g_force_oneshot{false};     // A/B switch (cloak_set_gemv_engine)
extern std::atomic<bool> g_gemv_pdl;                 // gemv_stream.cu

static cloak_status gemv_device(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y, uint32_t batch,
                                cudaStream_t s) {
    GemvArgs a;
    a.pool = pool->base;
    a.T = pool->d_T;
    a.log2b = pool->log2_block;
    a.w_offset = w->w_offset;
    a.N = w->N;
    a.K = w->K;
    a.x = d_x;
    a.y = d_y;
    a.batch = batch;
    a.zero = 0;
    if (!g_force_oneshot) {
        const int cu = gemv_stream_chunk(pool, w, batch);
        if (cu >= 1) {
            cloak_gemv_op op;
            op.w = *w;
            op.d_x = d_x;
            op.d_y = d_y;
            op.d_gate = nullptr;
            op.d_act = nullptr;
            op.after = 0;
            return gemv_stream_launch(pool, &op, 1, cu, batch, s);
        }
    }
    if (w->dt == CLOAK_BF16) {
        const uint32_t tiles = w->N / GV_ROWS;
        const uint32_t S = (w->K + GV_KCTA - 1) / GV_KCTA;
        float* part = nullptr;
        uint32_t* counters = nullptr;
        if (S > 1) {
            if (tiles > GV_MAX_TILES) return fail(CLOAK_ERR_UNSUPPORTED, "gemv: N too large for the split-K counters");
            const size_t need = WS_COUNTER_BYTES + (size_t)S * batch * w->N * 4;
            cloak_status st = pool_workspace(pool, need, s);
            if (st != CLOAK_OK) return st;
            counters = reinterpret_cast<uint32_t*>(pool->ws);
            part = reinterpret_cast<float*>(pool->ws + WS_COUNTER_BYTES);
        }
        const bool full = w->K % GV_KCTA == 0;
        const dim3 grid(tiles * S), blk(GV_WARPS * 32);
        if (batch <= 8) {
            if (full) gemv_bf16_kernel<1, true><<<grid, blk, 0, s>>>(a, S, part, counters);
            else      gemv_bf16_kernel<1, false><<<grid, blk, 0, s>>>(a, S, part, counters);
        } else {
            if (full) gemv_bf16_kernel<2, true><<<grid, blk, 0, s>>>(a, S, part, counters);
            else      gemv_bf16_kernel<2, false><<<grid, blk, 0, s>>>(a, S, part, counters);
        }
        launched();
    } else {
        const unsigned ctas = (w->N + 7) / 8;
        if (batch <= 4) gemv_f32_kernel<4><<<ctas, 256, 0, s>>>(a);
        else            gemv_f32_kernel<16><<<ctas, 256, 0, s>>>(a);
        launched();
    }
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

static cloak_status gemv_check(const cloak_pool* pool, const cloak_tensor* w, const void* x, void* y, uint32_t batch,
                               const char* who) {
    cloak_status st = check_linear(pool, w, x, y, who);
    if (st != CLOAK_OK) return st;
    if (batch < 1 || batch > 16) return fail(CLOAK_ERR_INVALID, "%s: batch must be in 1..16", who);
    if (w->layout != CLOAK_ROWMAJOR) return fail(CLOAK_ERR_UNSUPPORTED, "%s: only CLOAK_ROWMAJOR is implemented", who);
    if (w->dt == CLOAK_BF16) {
        if (w->K % 64 || w->N % 16) return fail(CLOAK_ERR_ALIGN, "%s: bf16 needs K %% 64 == 0 and N %% 16 == 0", who);
        if (pool->block < 128) return fail(CLOAK_ERR_UNSUPPORTED, "%s: bf16 needs block_bytes >= 128", who);
    } else if (w->K % 4) {
        return fail(CLOAK_ERR_ALIGN, "%s: f32 needs K %% 4 == 0", who);
    }
    return CLOAK_OK;
}

}  // namespace cloak

using namespace cloak;

namespace cloak { extern std::atomic<bool> g_gemv_exclusive; void gemv_set_fusion(bool on); }
extern "C" cloak_status cloak_set_gemv_engine(int engine) {
    if (engine < 0 || engine > 4) return fail(CLOAK_ERR_INVALID, "set_gemv_engine: engine must be 0 .. 4");
    g_force_oneshot = engine == 1;
    g_gemv_pdl = engine != 2;
    g_gemv_exclusive = engine == 3;
    gemv_set_fusion(engine != 4);
    return CLOAK_OK;
}

namespace cloak { extern std::atomic<unsigned long long*> g_trace; }
extern "C" cloak_status cloak_set_trace(void* d_trace) {
    if ((uintptr_t)d_trace & 7) return fail(CLOAK_ERR_ALIGN, "set_trace: buffer must be 8-byte aligned");
    g_trace.store(static_cast<unsigned long long*>(d_trace));
    return CLOAK_OK;
}

extern "C" cloak_status cloak_gemv(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                                   uint32_t batch, void* stream) {
    cloak_status st = gemv_check(pool, w, d_x, d_y, batch, "gemv");
    if (st != CLOAK_OK) return st;
    DeviceGuard g(pool->device);
    return gemv_device(pool, w, d_x, d_y, batch, (cudaStream_t)stream);
}

extern "C" cloak_status cloak_gemv_chain(const cloak_pool* pool, const cloak_gemv_op* h_ops, uint32_t n_ops, uint32_t batch,
                                         void* stream) {
    if (!h_ops || n_ops == 0) return fail(CLOAK_ERR_INVALID, "gemv_chain: no ops");
    std::vector<int> cb(n_ops);
    for (uint32_t i = 0; i < n_ops; ++i) {
        cloak_status st = gemv_check(pool, &h_ops[i].w, h_ops[i].d_x, h_ops[i].d_y, batch, "gemv_chain");
        if (st != CLOAK_OK) return st;
        if ((h_ops[i].d_gate == nullptr) != (h_ops[i].d_act == nullptr))
            return fail(CLOAK_ERR_INVALID, "gemv_chain: op %u: d_gate and d_act go together", i);
        if (h_ops[i].d_gate)                       // written by an earlier op?  then by one of the same shape
            for (uint32_t k = 0; k < i; ++k)
                if (h_ops[k].d_y == h_ops[i].d_gate && (h_ops[k].w.N != h_ops[i].w.N || h_ops[k].w.K != h_ops[i].w.K))
                    return fail(CLOAK_ERR_INVALID, "gemv_chain: op %u: d_gate is the output of op %u, which has another shape", i, k);
        cb[i] = gemv_stream_chunk(pool, &h_ops[i].w, batch);
        if (cb[i] < 1) return fail(CLOAK_ERR_UNSUPPORTED, "gemv_chain: op %u needs bf16 ROWMAJOR, K %% 256 == 0, block >= 512", i);
    }
    DeviceGuard g(pool->device);
    // consecutive ops with one chunk size, at most 48 at a time and within the row-tile counters, share a launch
    uint32_t i = 0;
    while (i < n_ops) {
        uint32_t n = 1;
        uint64_t tiles = h_ops[i].w.N / 8;
        while (i + n < n_ops && n < 48 && cb[i + n] == cb[i] && tiles + h_ops[i + n].w.N / 8 <= 200000) {
            tiles += h_ops[i + n].w.N / 8;
            ++n;
        }
        cloak_status st = gemv_stream_launch(pool, h_ops + i, n, cb[i], batch, (cudaStream_t)stream);
        if (st != CLOAK_OK) return st;
        i += n;
    }
    return CLOAK_OK;
}

// Host-buffer form of cloak_gemv_chain for independent ops: every op's d_x / d_y are HOST pointers.  All X go up, the chain
// runs, all Y come back; the stream is synchronised ONCE (cloak_gemv_host does that per projection).
extern "C" cloak_status cloak_gemv_chain_host(const cloak_pool* pool, const cloak_gemv_op* h_ops, uint32_t n_ops, uint32_t batch,
                                              void* stream) {
    if (!h_ops || n_ops == 0) return fail(CLOAK_ERR_INVALID, "gemv_chain_host: no ops");
    size_t total = 0;
    std::vector<size_t> xo(n_ops), yo(n_ops);
    for (uint32_t i = 0; i < n_ops; ++i) {
        cloak_status st = gemv_check(pool, &h_ops[i].w, h_ops[i].d_x, h_ops[i].d_y, batch, "gemv_chain_host");
        if (st != CLOAK_OK) return st;
        if (h_ops[i].d_gate || h_ops[i].d_act || h_ops[i].after)
            return fail(CLOAK_ERR_INVALID, "gemv_chain_host: op %u: ops must be independent (no d_gate / d_act / after)", i);
        const size_t e = h_ops[i].w.dt == CLOAK_F32 ? 4 : 2;
        xo[i] = total;
        total += ((size_t)batch * h_ops[i].w.K * e + 255) & ~(size_t)255;
        yo[i] = total;
        total += ((size_t)batch * h_ops[i].w.N * e + 255) & ~(size_t)255;
    }
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    AsyncBuf buf(s);
    if (cloak_status ast = buf.alloc(total)) return ast;
    char* d = static_cast<char*>(buf.p);
    std::vector<cloak_gemv_op> ops(h_ops, h_ops + n_ops);
    for (uint32_t i = 0; i < n_ops; ++i) {
        const size_t e = ops[i].w.dt == CLOAK_F32 ? 4 : 2;
        CLOAK_CUDA(cudaMemcpyAsync(d + xo[i], h_ops[i].d_x, (size_t)batch * ops[i].w.K * e, cudaMemcpyHostToDevice, s));
        ops[i].d_x = d + xo[i];
        ops[i].d_y = d + yo[i];
    }
    bool all_stream = !g_force_oneshot.load(std::memory_order_relaxed);
    for (uint32_t i = 0; i < n_ops && all_stream; ++i) all_stream = gemv_stream_chunk(pool, &ops[i].w, batch) >= 1;
    cloak_status st = CLOAK_OK;
    if (all_stream) {
        st = cloak_gemv_chain(pool, ops.data(), n_ops, batch, stream);
    } else {
        for (uint32_t i = 0; i < n_ops && st == CLOAK_OK; ++i) st = gemv_device(pool, &ops[i].w, ops[i].d_x, ops[i].d_y, batch, s);
    }
    if (st != CLOAK_OK) return st;
    for (uint32_t i = 0; i < n_ops; ++i) {
        const size_t e = ops[i].w.dt == CLOAK_F32 ? 4 : 2;
        CLOAK_CUDA(cudaMemcpyAsync(h_ops[i].d_y, d + yo[i], (size_t)batch * ops[i].w.N * e, cudaMemcpyDeviceToHost, s));
    }
    CLOAK_CUDA(cudaStreamSynchronize(s));
    return CLOAK_OK;
}

extern "C" cloak_status cloak_gemv_chain_scratch_bytes(const cloak_pool* pool, const cloak_gemv_op* h_ops, uint32_t n_ops,
                                                       uint32_t batch, uint64_t* h_bytes) {
    if (!h_ops || n_ops == 0 || !h_bytes) return fail(CLOAK_ERR_INVALID, "gemv_chain_scratch_bytes: NULL argument or no ops");
    uint64_t need = 0;
    const uint64_t sms = (uint64_t)sm_count(pool ? pool->device : 0);
    for (uint32_t i = 0; i < n_ops; ++i) {
        const cloak_tensor& w = h_ops[i].w;
        cloak_status st = gemv_check(pool, &w, h_ops[i].d_x, h_ops[i].d_y, batch, "gemv_chain_scratch_bytes");
        if (st != CLOAK_OK) return st;
        uint64_t b = 0;
        if (!g_force_oneshot.load(std::memory_order_relaxed) && gemv_stream_chunk(pool, &w, batch) >= 1)
            b = WS_COUNTER_BYTES + 48ull * sms * batch * 8 * 4;          // a full launch of the streaming kernel: one cut-tile partial per (op, CTA)
        else if (w.dt == CLOAK_BF16 && (w.K + GV_KCTA - 1) / GV_KCTA > 1)
            b = WS_COUNTER_BYTES + (uint64_t)((w.K + GV_KCTA - 1) / GV_KCTA) * batch * w.N * 4;
        if (b > need) need = b;
    }
    *h_bytes = need;
    return CLOAK_OK;
}

extern "C" cloak_status cloak_gemv_host(const cloak_pool* pool, const cloak_tensor* w, const void* h_x, void* h_y,
                                        uint32_t batch, void* stream) {
    cloak_status st = gemv_check(pool, w, h_x, h_y, batch, "gemv_host");
    if (st != CLOAK_OK) return st;
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t e = w->dt == CLOAK_F32 ? 4 : 2;
    const size_t xb = (size_t)batch * w->K * e, yb = (size_t)batch * w->N * e;
    const size_t xpad = (xb + 255) & ~(size_t)255;
    AsyncBuf buf(s);                            // from the library's cached pool: no driver allocation after the first call
    st = buf.alloc(xpad + yb);
    if (st != CLOAK_OK) return st;
    char* d = static_cast<char*>(buf.p);
    CLOAK_CUDA(cudaMemcpyAsync(d, h_x, xb, cudaMemcpyHostToDevice, s));
    st = gemv_device(pool, w, d, d + xpad, batch, s);
    if (st != CLOAK_OK) return st;
    CLOAK_CUDA(cudaMemcpyAsync(h_y, d + xpad, yb, cudaMemcpyDeviceToHost, s));
    CLOAK_CUDA(cudaStreamSynchronize(s));       // h_y is the caller's to read when the call returns
    return CLOAK_OK;
}
