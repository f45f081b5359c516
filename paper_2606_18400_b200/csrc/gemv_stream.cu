// S6 cloak_gemv, bf16, K % 256 == 0: the streaming (persistent, TMA-fed) kernel.
//
// Same contraction and table translation as gemv.cu (north_star (c)), organised for the
// HBM roofline.  Measured on B200: a pure stream of 16 x 2 KiB row pieces per stage tops out
// at 5.5 TB/s, 8 x 4 KiB pieces at 6.4 TB/s, so a unit of work is (8 weight rows) x (CB = 4 KiB of each row):
//   * one persistent CTA per SM; units are numbered tile-major (u = tile * kch + chunk) and cut into equal
//     contiguous ranges, one per CTA (stream-K): every SM moves the same bytes, no wave tail;
//   * warp 0 produces: 8 lanes each translate one row piece through the block table and issue one
//     cp.async.bulk (TMA 1-D) into a shared-memory ring (6 stages of 32 KiB), completion on an mbarrier;
//   * warps 1-8 consume: each owns one eighth of the k-range of a chunk.  The weights are the B operand of
//     mma.sync.m16n8k16 (8 weight rows = N), the activations the A operand (batch rows = M, zero-padded to 8 or
//     16).  Lane (g, t) reads one 16-byte vector of weight row g per 64-byte step; since a contraction may visit
//     k in any order, the vector's elements are *declared* to be the MMA's k-slots (2t, 2t+1, 2t+8, 2t+9) and
//     X is loaded by the same rule: both operands are plain 16-byte loads, no transposes;
//   * inside its range a CTA walks groups of TG = 8 row tiles chunk-major (all tiles of the group for chunk 0,
//     then chunk 1, ...), so a warp's X fragments are fetched once per (group, chunk) and reused for 64 weight
//     rows: X traffic from L2 is batch/64 of the weight traffic instead of batch/16 (at batch 16 the old
//     tile-major walk spent as many L2 bytes on X as on W);
//   * accumulators (one m16n8 tile per row tile of the group, two interleaved to halve the dependency chain)
//     stay in registers until the group is done, are reduced over the 8 warps in shared memory, and stored.
//     A row tile cut by a range boundary writes fp32 partials and the last contributor to arrive sums them in
//     contributor order: deterministic, and bit-identical between a cloaked and an identity-table pool, which
//     differ only in addresses.
//   * programmatic dependent launch: the grid may start while its stream predecessor drains; the producer
//     streams W (immutable during decode) ahead of griddepcontrol.wait, everything else waits.
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
    float* part;         // [tile][maxc][batch][8]
    uint32_t* counters;  // [tile], zero between launches
    uint32_t early;      // 1: W is unchanged since before the preceding kernel, so the producer may stream it
                         //    ahead of griddepcontrol.wait (programmatic dependent launch)
};

constexpr int GS_CONSUMERS = 8;                       // consumer warps
constexpr int GS_THREADS = 32 * (1 + GS_CONSUMERS);
constexpr int GS_ROWS = 8;                            // weight rows per tile (the MMA's N)
constexpr int GS_PAD = 64;                            // bytes of padding per staged row (conflict-free LDS.128)
// Row tiles per group (X reuse; one register accumulator set per tile) and interleaved accumulators per tile.
// 8 tiles x 2 accumulators measured best for both batch ranges: 16 x 1 halves the X traffic at batch 16 but its
// 16-deep dependent MMA chain costs more than that saves; staggering the group boundaries over the CTAs (so the
// SMs do not all wait for X at once) adds a group per CTA and was slower too.
constexpr int gs_tg(int nt) { return 8; }
constexpr int gs_nacc(int nt) { return 2; }
constexpr int GS_TGR = 4;                             // row tiles reduced across warps per shared-memory pass
constexpr int GS_MAX_STAGES = 12;
constexpr uint32_t gs_stages(int log2cb) {            // ~192 KiB of weights in flight per SM
    return (196608u >> (log2cb + 3)) > GS_MAX_STAGES ? GS_MAX_STAGES : (196608u >> (log2cb + 3));
}

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

// LOG2CB: log2 of the chunk bytes per row (9..12).  NT: 1 = batch <= 8 (upper half of the MMA's M is zero), 2 = batch <= 16.
template <int LOG2CB, int NT>
__global__ void __launch_bounds__(GS_THREADS, 1) gemv_stream_kernel(GemvStreamArgs a) {
    constexpr uint32_t CB = 1u << LOG2CB;
    constexpr uint32_t RS = CB + GS_PAD;                       // staged row stride
    constexpr uint32_t STAGE = GS_ROWS * RS;
    constexpr uint32_t NST = gs_stages(LOG2CB);
    constexpr int GS_TG = gs_tg(NT), NACC = gs_nacc(NT);
    constexpr int KS = CB / (GS_CONSUMERS * 64);               // 64-byte steps (one 16-byte vector per lane) per warp per unit
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full[NST], empty[NST];
    __shared__ float red[GS_CONSUMERS][GS_TGR][NT * 64];      // [warp][tile][batch m][row r]
    __shared__ uint32_t last_flag[2];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
#pragma unroll
        for (uint32_t s = 0; s < NST; ++s) {
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
    const uint32_t tile_lo = ubeg / a.kch, tile_hi = (uend - 1) / a.kch;

    if (warp == 0) {
        // ------------------------------------------------------------ producer
        // The table is immutable after cloak_pool_create; the weights may have been written by the preceding
        // kernel (a shuffle / re-layout) unless the host says otherwise.
        if (!a.early) grid_dep_wait();
        uint32_t s = 0, ph = 0;
        bool wrapped = false;
        for (uint32_t g0 = tile_lo; g0 <= tile_hi; g0 += GS_TG) {
            const uint32_t g1 = min(g0 + GS_TG - 1, tile_hi);
            for (uint32_t c = 0; c < a.kch; ++c) {
                for (uint32_t tile = g0; tile <= g1; ++tile) {
                    const uint32_t u = tile * a.kch + c;
                    if (u < ubeg || u >= uend) continue;
                    if (wrapped) mbar_wait(smem_u32(&empty[s]), ph ^ 1);
                    const uint32_t bar = smem_u32(&full[s]);
                    if (lane == 0) mbar_expect_tx(bar, GS_ROWS * CB);
                    __syncwarp();
                    if (lane < GS_ROWS) {
                        const uint64_t off = a.w_offset + ((uint64_t)(tile * GS_ROWS + lane) * a.K) * 2 + (uint64_t)c * CB;
                        const uint32_t slot = __ldg(a.T + (off >> a.log2b));
                        const char* src = a.pool + ((uint64_t)slot << a.log2b) + (off & ((1ull << a.log2b) - 1));
                        bulk_g2s(smem_base + s * STAGE + lane * RS, src, CB, bar);
                    }
                    if (++s == NST) { s = 0; ph ^= 1; wrapped = true; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    const int cw = warp - 1;
    const int g = lane >> 2, t = lane & 3;
    const uint32_t ctid = threadIdx.x - 32;                        // 0..255 among consumers
    const bool xv0 = (uint32_t)g < a.batch, xv1 = (uint32_t)(g + 8) < a.batch;
    const uint32_t lane_off = cw * (CB / GS_CONSUMERS) + t * 16;   // byte offset of this lane inside a row chunk
    const uint16_t* x0 = a.x + (size_t)g * a.K + lane_off / 2;
    const uint16_t* x1 = a.x + (size_t)(g + 8) * a.K + lane_off / 2;
    const uint32_t nout = a.batch * GS_ROWS;

    // X, Y, the split-K partials and counters all belong to stream order: nothing below touches them before the
    // predecessor has completed.  Meanwhile the producer is already filling the ring.
    grid_dep_wait();
    if (ctid == 0) grid_dep_launch();

    auto is_cut = [&](uint32_t tile) {       // does a range boundary cut this row tile?
        return (tile == tile_lo && ubeg > tile * a.kch) || (tile == tile_hi && uend < (tile + 1) * a.kch);
    };

    uint32_t s = 0, ph = 0;
    for (uint32_t g0 = tile_lo; g0 <= tile_hi; g0 += GS_TG) {
        const uint32_t g1 = min(g0 + GS_TG - 1, tile_hi);
        float acc[GS_TG][NACC][4];
#pragma unroll
        for (int j = 0; j < GS_TG; ++j)
#pragma unroll
            for (int n = 0; n < NACC; ++n)
#pragma unroll
                for (int i = 0; i < 4; ++i) acc[j][n][i] = 0.f;

        for (uint32_t c = 0; c < a.kch; ++c) {
            // this warp's X fragments for chunk c: fetched once, reused for every row tile of the group
            uint4 xa[KS], xb[KS];
            const uint32_t xk = c * (CB / 2);
            const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                xa[ks] = xv0 ? __ldg(reinterpret_cast<const uint4*>(x0 + xk + ks * 32)) : z;
                xb[ks] = (NT == 2 && xv1) ? __ldg(reinterpret_cast<const uint4*>(x1 + xk + ks * 32)) : z;
            }
#pragma unroll
            for (int j = 0; j < GS_TG; ++j) {
                const uint32_t tile = g0 + j, u = tile * a.kch + c;
                if (tile > g1 || u < ubeg || u >= uend) continue;
                mbar_wait(smem_u32(&full[s]), ph);
                const uint32_t base = smem_base + s * STAGE + g * RS + lane_off;
#pragma unroll
                for (int ks = 0; ks < KS; ++ks) {
                    const uint4 w = lds128(base + ks * 64);
                    mma_16816(acc[j][0], xa[ks].x, xb[ks].x, xa[ks].y, xb[ks].y, w.x, w.y);
                    mma_16816(acc[j][NACC - 1], xa[ks].z, xb[ks].z, xa[ks].w, xb[ks].w, w.z, w.w);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&empty[s]));
                if (++s == NST) { s = 0; ph ^= 1; }
            }
        }

        // ---- the group is done: reduce over the 8 warps (each summed its own k-slice), GS_TGR row tiles per pass
#pragma unroll
        for (int sb = 0; sb < GS_TG / GS_TGR; ++sb) {
            const uint32_t tb = g0 + sb * GS_TGR;
            if (tb <= g1) {
#pragma unroll
                for (int jj = 0; jj < GS_TGR; ++jj) {
                    const int j = sb * GS_TGR + jj;
                    float* r = red[cw][jj];
                    float v[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) v[i] = NACC == 2 ? acc[j][0][i] + acc[j][NACC - 1][i] : acc[j][0][i];
                    r[g * 8 + 2 * t] = v[0];
                    r[g * 8 + 2 * t + 1] = v[1];
                    if (NT == 2) {
                        r[(g + 8) * 8 + 2 * t] = v[2];
                        r[(g + 8) * 8 + 2 * t + 1] = v[3];
                    }
                }
                consumer_bar();
                for (uint32_t o = ctid; o < GS_TGR * NT * 64; o += GS_CONSUMERS * 32) {
                    const uint32_t jj = o / (NT * 64), rem = o % (NT * 64), m = rem / 8, r = rem % 8;
                    const uint32_t tile = tb + jj;
                    if (tile > g1 || m >= a.batch) continue;
                    float sum = red[0][jj][rem];
#pragma unroll
                    for (int w = 1; w < GS_CONSUMERS; ++w) sum += red[w][jj][rem];
                    if (!is_cut(tile)) {
                        a.y[(size_t)m * a.N + tile * GS_ROWS + r] = __float2bfloat16_rn(sum);
                    } else {
                        const uint32_t me = blockIdx.x - (tile * a.kch) / a.per;
                        __stcg(a.part + ((size_t)tile * a.maxc + me) * nout + m * GS_ROWS + r, sum);
                    }
                }
                consumer_bar();      // red[] is reused by the next pass
            }
        }
    }

    // ---- row tiles cut by a range boundary (at most the first and the last of the range): their partials were
    // written above; publish them once, at the end, and let the last contributor to arrive sum them in order.
    const bool cut_lo = is_cut(tile_lo), cut_hi = tile_hi != tile_lo && is_cut(tile_hi);
    if (cut_lo || cut_hi) {
        __threadfence();
        consumer_bar();
        if (ctid < 2) {
            const uint32_t tile = ctid == 0 ? tile_lo : tile_hi;
            uint32_t flag = 0;
            if (ctid == 0 ? cut_lo : cut_hi) {
                const uint32_t ncontrib = (tile * a.kch + a.kch - 1) / a.per - (tile * a.kch) / a.per + 1;
                const uint32_t old = atomicAdd(a.counters + tile, 1u);
                if (old == ncontrib - 1) {
                    a.counters[tile] = 0;               // self-reset for the next launch
                    flag = ncontrib;
                }
            }
            last_flag[ctid] = flag;
        }
        consumer_bar();
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const uint32_t nc = last_flag[e];
            if (nc == 0) continue;
            __threadfence();
            const uint32_t tile = e == 0 ? tile_lo : tile_hi;
            const float* base = a.part + (size_t)tile * a.maxc * nout;
            for (uint32_t i = ctid; i < nout; i += GS_CONSUMERS * 32) {
                float sum = 0.f;
                for (uint32_t q = 0; q < nc; ++q) sum += __ldcg(base + (size_t)q * nout + i);
                a.y[(size_t)(i / GS_ROWS) * a.N + tile * GS_ROWS + (i % GS_ROWS)] = __float2bfloat16_rn(sum);
            }
        }
    }
}

bool g_gemv_pdl = true;      // A/B switch (cloak_set_gemv_engine(2) turns PDL off)

template <int LOG2CB, int NT>
static cloak_status launch(const GemvStreamArgs& a, int ctas, cudaStream_t s) {
    constexpr size_t smem = (size_t)gs_stages(LOG2CB) * GS_ROWS * ((1u << LOG2CB) + GS_PAD);
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
    return CLOAK_OK;
}

// Entry used by gemv.cu.  Preconditions (checked there): bf16, ROWMAJOR, K % 256 == 0, N % 16 == 0, block >= 512 B.
cloak_status gemv_stream_bf16(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y, uint32_t batch,
                              cudaStream_t s) {
    const uint64_t row_bytes = (uint64_t)w->K * 2;
    int log2cb = 12;
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
        case 12: return nt2 ? launch<12, 2>(a, ctas, s) : launch<12, 1>(a, ctas, s);
        case 11: return nt2 ? launch<11, 2>(a, ctas, s) : launch<11, 1>(a, ctas, s);
        case 10: return nt2 ? launch<10, 2>(a, ctas, s) : launch<10, 1>(a, ctas, s);
        default: return nt2 ? launch<9, 2>(a, ctas, s) : launch<9, 1>(a, ctas, s);
    }
}

}  // namespace cloak
