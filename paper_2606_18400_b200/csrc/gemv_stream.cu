// S6 cloak_gemv, bf16, K % 256 == 0: the streaming (persistent, TMA-fed) kernel.
//
// Same contraction and table translation as gemv.cu (north_star (c)), organised for the
// HBM roofline:
//   * one persistent CTA per SM; the (row tile of 16 rows) x (k chunk of CB bytes per row) "units" of the
//     matrix are numbered tile-major and cut into equal contiguous ranges, one per CTA (stream-K), so every
//     SM moves the same number of bytes and there is no wave tail;
//   * warp 0 is the producer: for each unit, 16 lanes each translate one row chunk through the block table
//     and issue one cp.async.bulk (TMA 1-D) of CB bytes into a 6-stage shared-memory ring, completion on an
//     mbarrier -- ~190 KiB in flight per SM all the time, no registers or LSU slots spent on weight bytes;
//   * warps 1-4 consume: a quarter of the chunk each, 16-byte LDS in the k-permuted fragment order of
//     gemv.cu (rows padded by 64 B -> conflict-free), mma.sync.m16n8k16 bf16 with the batch as N;
//   * accumulators stay in registers across the units of a tile.  A tile wholly inside one CTA's range is
//     reduced over the 4 warps in shared memory and stored; a tile cut by a range boundary writes fp32
//     partials and the last contributor to arrive sums them in contributor order (deterministic, and
//     identical for a cloaked and an identity-table pool, which only differ in addresses).
#include <cuda_bf16.h>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

struct GemvStreamArgs {
    const char* pool;
    const uint32_t* T;
    uint32_t log2b;
    uint64_t w_offset;
    uint32_t N, K;
    const uint16_t* x;
    __nv_bfloat16* y;
    uint32_t batch;
    uint32_t kch;        // chunks per row = K*2 / CB
    uint32_t units;      // tiles * kch
    uint32_t per;        // units per CTA
    uint32_t maxc;       // max contributors per tile
    float* part;         // [tile][maxc][batch][16]
    uint32_t* counters;  // [tile], zero between launches
    uint32_t early;      // 1: W is unchanged since before the preceding kernel, so the producer may stream it
                         //    ahead of griddepcontrol.wait (programmatic dependent launch)
};

constexpr int GS_STAGES = 6;
constexpr int GS_CONSUMERS = 4;                       // consumer warps
constexpr int GS_THREADS = 32 * (1 + GS_CONSUMERS);
constexpr int GS_ROWS = 16;
constexpr int GS_PAD = 64;                            // bytes of padding per staged row

__device__ __forceinline__ void mma_16816(float c[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                          uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}
// Programmatic dependent launch (PDL): this grid may start while its stream predecessor is still draining.
// grid_dep_wait returns once the predecessor has completed and its writes are visible; grid_dep_launch lets the
// stream successor start.  Every kernel here triggers only AFTER its own wait, so whatever a successor does ahead
// of its wait still observes everything older than its immediate predecessor.
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" :: "n"(GS_CONSUMERS * 32) : "memory"); }

// LOG2CB: log2 of the chunk bytes per row (9, 10 or 11).  NT: 8-wide batch tiles.
template <int LOG2CB, int NT>
__global__ void __launch_bounds__(GS_THREADS, 1) gemv_stream_kernel(GemvStreamArgs a) {
    constexpr uint32_t CB = 1u << LOG2CB;
    constexpr uint32_t RS = CB + GS_PAD;                       // staged row stride
    constexpr uint32_t STAGE = GS_ROWS * RS;
    constexpr int KS = CB / (GS_CONSUMERS * 128);              // 128-byte k-steps per consumer warp per unit
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full[GS_STAGES], empty[GS_STAGES];
    __shared__ float red[GS_CONSUMERS][NT * 8][GS_ROWS + 1];
    __shared__ uint32_t last_flag;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < GS_STAGES; ++s) {
            mbar_init(smem_u32(&full[s]), 1);
            mbar_init(smem_u32(&empty[s]), GS_CONSUMERS);
        }
        fence_barrier_init();
    }
    __syncthreads();

    const uint32_t ubeg = blockIdx.x * a.per;
    const uint32_t uend = min(ubeg + a.per, a.units);
    if (ubeg >= uend) return;
    const uint32_t smem_base = smem_u32(smem);

    if (warp == 0) {
        // ------------------------------------------------------------ producer
        // The table is immutable after cloak_pool_create; the weights may have been written by the preceding
        // kernel (a shuffle / re-layout) unless the host says otherwise.
        if (!a.early) grid_dep_wait();
        uint32_t it = 0;
        for (uint32_t u = ubeg; u < uend; ++u, ++it) {
            const uint32_t s = it % GS_STAGES, f = it / GS_STAGES;
            if (f > 0) mbar_wait(smem_u32(&empty[s]), (f - 1) & 1);
            const uint32_t tile = u / a.kch, c = u - tile * a.kch;
            const uint32_t bar = smem_u32(&full[s]);
            if (lane == 0) mbar_expect_tx(bar, GS_ROWS * CB);
            __syncwarp();
            if (lane < GS_ROWS) {
                const uint64_t off = a.w_offset + ((uint64_t)(tile * GS_ROWS + lane) * a.K) * 2 + (uint64_t)c * CB;
                const uint32_t slot = __ldg(a.T + (off >> a.log2b));
                const char* src = a.pool + ((uint64_t)slot << a.log2b) + (off & ((1ull << a.log2b) - 1));
                bulk_g2s(smem_base + s * STAGE + lane * RS, src, CB, bar);
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    const int cw = warp - 1;
    const int g = lane >> 2, t = lane & 3;
    const int ctid = threadIdx.x - 32;                              // 0..127 among consumers
    const bool xv0 = (uint32_t)g < a.batch, xv1 = (uint32_t)(g + 8) < a.batch;
    const uint32_t lane_off = cw * (CB / GS_CONSUMERS) + t * 16;     // byte offset of this lane inside a row chunk
    const uint16_t* x0 = a.x + (size_t)g * a.K + lane_off / 2;
    const uint16_t* x1 = a.x + (size_t)(g + 8) * a.K + lane_off / 2;

    float acc[NT][4];
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

    // X, Y, the split-K partials and counters all belong to stream order: nothing below touches them before the
    // predecessor has completed.  Meanwhile the producer is already filling the ring.
    grid_dep_wait();
    if (ctid == 0) grid_dep_launch();

    auto flush = [&](uint32_t tile, uint32_t u_first, uint32_t u_last) {
        // u_first / u_last: the units of `tile` this CTA has accumulated (inclusive range)
#pragma unroll
        for (int i = 0; i < NT; ++i) {
            red[cw][i * 8 + 2 * t][g] = acc[i][0];
            red[cw][i * 8 + 2 * t + 1][g] = acc[i][1];
            red[cw][i * 8 + 2 * t][g + 8] = acc[i][2];
            red[cw][i * 8 + 2 * t + 1][g + 8] = acc[i][3];
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
        }
        consumer_bar();
        const uint32_t nout = a.batch * GS_ROWS;
        const uint32_t t_first = tile * a.kch, t_last = t_first + a.kch - 1;
        const uint32_t n0 = tile * GS_ROWS;
        if (u_first == t_first && u_last == t_last) {
            for (uint32_t i = ctid; i < nout; i += GS_CONSUMERS * 32) {
                const uint32_t m = i / GS_ROWS, r = i % GS_ROWS;
                float s = red[0][m][r];
#pragma unroll
                for (int w = 1; w < GS_CONSUMERS; ++w) s += red[w][m][r];
                a.y[(size_t)m * a.N + n0 + r] = __float2bfloat16_rn(s);
            }
        } else {
            const uint32_t c_first = t_first / a.per, c_last = t_last / a.per;
            const uint32_t ncontrib = c_last - c_first + 1, me = blockIdx.x - c_first;
            float* mine = a.part + ((size_t)tile * a.maxc + me) * nout;
            for (uint32_t i = ctid; i < nout; i += GS_CONSUMERS * 32) {
                const uint32_t m = i / GS_ROWS, r = i % GS_ROWS;
                float s = red[0][m][r];
#pragma unroll
                for (int w = 1; w < GS_CONSUMERS; ++w) s += red[w][m][r];
                __stcg(mine + i, s);
            }
            __threadfence();
            consumer_bar();
            if (ctid == 0) {
                const uint32_t old = atomicAdd(a.counters + tile, 1u);
                last_flag = (old == ncontrib - 1);
                if (old == ncontrib - 1) a.counters[tile] = 0;      // self-reset for the next launch
            }
            consumer_bar();
            if (last_flag) {
                __threadfence();
                const float* base = a.part + (size_t)tile * a.maxc * nout;
                for (uint32_t i = ctid; i < nout; i += GS_CONSUMERS * 32) {
                    const uint32_t m = i / GS_ROWS, r = i % GS_ROWS;
                    float s = 0.f;
                    for (uint32_t q = 0; q < ncontrib; ++q) s += __ldcg(base + (size_t)q * nout + i);
                    a.y[(size_t)m * a.N + n0 + r] = __float2bfloat16_rn(s);
                }
            }
        }
        consumer_bar();      // red[] and last_flag are reused by the next tile
    };

    // Activations of one unit: this lane's 16-byte vectors of X rows g (and g+8).  They come from L2 (X is up to
    // 16 x K x 2 bytes, more than the L1 left beside the ring), so the next unit's are fetched before this unit's
    // weights are waited for: their latency hides behind the LDS/MMA work.
    uint4 xa[KS][2], xb[KS][2], na[KS][2], nb[KS][2];
    auto load_x = [&](uint4 (&pa)[KS][2], uint4 (&pb)[KS][2], uint32_t c) {
        const uint32_t xk = c * (CB / 2);
        const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                pa[ks][h] = xv0 ? __ldg(reinterpret_cast<const uint4*>(x0 + xk + ks * 64 + h * 32)) : z;
                if (NT == 2) pb[ks][h] = xv1 ? __ldg(reinterpret_cast<const uint4*>(x1 + xk + ks * 64 + h * 32)) : z;
            }
    };
    load_x(xa, xb, ubeg % a.kch);

    uint32_t cur_tile = ubeg / a.kch, tile_first_u = ubeg;
    uint32_t it = 0;
    for (uint32_t u = ubeg; u < uend; ++u, ++it) {
        const uint32_t tile = u / a.kch;
        if (tile != cur_tile) {
            flush(cur_tile, tile_first_u, u - 1);
            cur_tile = tile;
            tile_first_u = u;
        }
        if (u + 1 < uend) load_x(na, nb, (u + 1) % a.kch);
        const uint32_t s = it % GS_STAGES, f = it / GS_STAGES;
        mbar_wait(smem_u32(&full[s]), f & 1);
        const uint32_t lo = smem_base + s * STAGE + g * RS + lane_off;
        const uint32_t hi = lo + 8 * RS;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const uint4 wl = lds128(lo + ks * 128 + h * 64);
                const uint4 wh = lds128(hi + ks * 128 + h * 64);
                mma_16816(acc[0], wl.x, wh.x, wl.y, wh.y, xa[ks][h].x, xa[ks][h].y);
                mma_16816(acc[0], wl.z, wh.z, wl.w, wh.w, xa[ks][h].z, xa[ks][h].w);
                if (NT == 2) {
                    mma_16816(acc[1], wl.x, wh.x, wl.y, wh.y, xb[ks][h].x, xb[ks][h].y);
                    mma_16816(acc[1], wl.z, wh.z, wl.w, wh.w, xb[ks][h].z, xb[ks][h].w);
                }
            }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&empty[s]));
#pragma unroll
        for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                xa[ks][h] = na[ks][h];
                if (NT == 2) xb[ks][h] = nb[ks][h];
            }
    }
    flush(cur_tile, tile_first_u, uend - 1);
}

bool g_gemv_pdl = true;      // A/B switch (cloak_set_gemv_engine(2) turns PDL off)

template <int LOG2CB, int NT>
static cloak_status launch(const GemvStreamArgs& a, int ctas, cudaStream_t s) {
    constexpr size_t smem = (size_t)GS_STAGES * GS_ROWS * ((1u << LOG2CB) + GS_PAD);
    static bool attr_set = false;
    if (!attr_set) {
        CLOAK_CUDA(cudaFuncSetAttribute(gemv_stream_kernel<LOG2CB, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ctas);
    cfg.blockDim = dim3(GS_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = g_gemv_pdl ? 1 : 0;
    CLOAK_CUDA(cudaLaunchKernelEx(&cfg, gemv_stream_kernel<LOG2CB, NT>, a));
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

// Entry used by gemv.cu.  Preconditions (checked there): bf16, ROWMAJOR, K % 256 == 0, N % 16 == 0, block >= 512 B.
cloak_status gemv_stream_bf16(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y, uint32_t batch,
                              cudaStream_t s) {
    const uint64_t row_bytes = (uint64_t)w->K * 2;
    int log2cb = 11;
    while (log2cb > 9 && (row_bytes & ((1u << log2cb) - 1))) --log2cb;
    if ((uint32_t)log2cb > pool->log2_block) log2cb = (int)pool->log2_block;
    if (log2cb < 9 || (row_bytes & ((1u << log2cb) - 1))) return fail(CLOAK_ERR_UNSUPPORTED, "gemv_stream: K*2 not a multiple of 512");
    GemvStreamArgs a;
    a.pool = pool->base;
    a.T = pool->d_T;
    a.log2b = pool->log2_block;
    a.w_offset = w->w_offset;
    a.N = w->N;
    a.K = w->K;
    a.x = static_cast<const uint16_t*>(d_x);
    a.y = static_cast<__nv_bfloat16*>(d_y);
    a.batch = batch;
    a.kch = (uint32_t)(row_bytes >> log2cb);
    const uint32_t tiles = w->N / GS_ROWS;
    const uint64_t units64 = (uint64_t)tiles * a.kch;
    if (units64 > 0xffffffffull) return fail(CLOAK_ERR_UNSUPPORTED, "gemv_stream: tensor too large");
    a.units = (uint32_t)units64;
    const int sms = sm_count(pool->device);
    a.per = (a.units + sms - 1) / sms;
    const int ctas = (int)((a.units + a.per - 1) / a.per);
    a.maxc = (a.kch + a.per - 1) / a.per + 1;
    const size_t need = WS_COUNTER_BYTES + (size_t)tiles * a.maxc * batch * GS_ROWS * 4;
    if ((size_t)tiles * 4 > WS_COUNTER_BYTES) return fail(CLOAK_ERR_UNSUPPORTED, "gemv_stream: N too large for the tile counters");
    cloak_status st = pool_workspace(pool, need);
    if (st != CLOAK_OK) return st;
    a.counters = reinterpret_cast<uint32_t*>(pool->ws);
    a.part = reinterpret_cast<float*>(pool->ws + WS_COUNTER_BYTES);
    a.early = (g_gemv_pdl && !pool->dirty) ? 1u : 0u;
    if (pool->dirty && pool->dirty_stream == s) pool->dirty = false;   // this launch waits for the writer in full
    const bool nt2 = batch > 8;
    switch (log2cb) {
        case 11: return nt2 ? launch<11, 2>(a, ctas, s) : launch<11, 1>(a, ctas, s);
        case 10: return nt2 ? launch<10, 2>(a, ctas, s) : launch<10, 1>(a, ctas, s);
        default: return nt2 ? launch<9, 2>(a, ctas, s) : launch<9, 1>(a, ctas, s);
    }
}

}  // namespace cloak
