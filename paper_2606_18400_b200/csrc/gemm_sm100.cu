// S7 cloak_gemm: batch 1..256 (MMA columns rounded up to 16) contraction on tcgen05 tensor cores, W tiles fetched by TMA through the table.
//
// Definition (north_star (c) "batch>1 gather-fused GEMM ... tcgen05/TMEM tiles fed by TMA through
// the permutation table"; BASELINE.json configs[3]):  Y[m, n] = sum_k X[m, k] * W[n, k], W in CLOAK_TILE128
// storage (tile (tn,tk) of 128x128 bf16 = 32 KiB contiguous, row-major inside), block_bytes >= 32 KiB.
//
// Mapping to the hardware.
//   * The pool is ONE 2-D TMA tensor map: rows of 128 bf16 (256 B).  Tile index i of the tensor sits at arena
//     byte w_offset + i*32 KiB = pool byte (T[blk] << log2 b) + within, i.e. at map row that/256: the permutation
//     enters only as a TMA coordinate.  A tile is fetched as two boxes of [128 rows x 64 cols] with
//     SWIZZLE_128B, which land in shared memory in the canonical K-major UMMA layout (8-row atoms of 1 KiB).
//   * A operand = the W tile (M = 128 output features), B operand = X[batch, 64] boxes of a second map over X
//     (N = batch), D = 128 lanes x batch fp32 columns in TMEM, two accumulator buffers.
//   * Units = tiles, numbered tn-major (= TILE128 storage order), the ops of a launch back to back: ONE sequence per
//     launch, cut into CHUNKS.  The kernel is HBM-bound (AI = batch flop/B < ridge), so what matters is that every SM
//     streams with a full TMA ring until the last byte of the launch has arrived -- and the SMs do not stream equally
//     fast (with equal shares the fastest SM finished at 70 % of the launch, the mean at 81 %: ncu,
//     profiles/r1_ncu_full_gemm_b32.md).  So a CTA first takes a static chunk (a share of ~3/4 of the equal split), then
//     pulls small chunks from the rest of the sequence off an atomic counter until it is empty.
//   * Roles: warp 0 = scheduler + TMA producer for W (one lane), warp 1 = MMA issuer (one lane) + TMEM allocator,
//     warp 2 = TMA producer for X (own shallow ring), warps 3-6 = epilogue (tcgen05.ld 32x32b, one TMEM lane quarter
//     each).  The scheduler hands every chunk to the other roles through a small shared-memory queue.
//   * A tile row wholly inside a chunk is stored as bf16 straight from TMEM.  A row cut by chunk boundaries has
//     contributors: each takes a ticket; all but the holder of the last ticket write fp32 partials, the last one adds
//     them to its own accumulator IN CHUNK ORDER as it drains it.  The chunk grid is fixed by the shapes, only the
//     assignment of chunks to CTAs varies, so the result does not depend on the schedule (deterministic; identical for
//     cloaked and identity-table pools).
//   * Row groups (GemmArgs::nacc = 2 in long launches, see gemm_grouping): a unit is then one k step of TWO adjacent tile
//     rows -- two weight tiles, ONE X tile, two MMAs per X stage into two accumulators (4 x batch TMEM columns with the
//     double buffer) -- which halves the X traffic from L2 (xbar2l1tex 1.96 x W -> 1.51 x W) and is worth 8-10 % at batch
//     32 .. 128; the schedule then runs over pair rows, tickets and partials stay per real tile row.
//   * Measured and dropped in round 1: a `cta_group::2` CTA-pair variant (M = 256 over two tile rows, each CTA loading half
//     of X) on the then static schedule: correct and no faster (1.53 vs 1.51 ms for 8 layers of cfg3).
#include <cuda_bf16.h>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

constexpr int GM_MAX_OPS = 16;             // ops per launch (one X tensor map of 128 B each in the kernel parameters)

struct GemmOp {
    uint64_t w_offset;
    __nv_bfloat16* y;
    uint32_t N;
    uint32_t kt;         // k tiles per tile row = K/128
    uint32_t units;      // (N/128) * kt
    uint32_t ubase;      // this op's first unit in the launch's unit sequence (ops back to back)
    uint32_t row_base;   // index of this op's first tile row among the launch's tile rows (tickets, ready counters)
    uint32_t dyn_row0;   // first tile row of this op in the dynamic part (N/128 if none)
    uint32_t pieces;     // dynamic part: chunks per tile row, each plen tiles (the last one the rest)
    uint32_t plen;
    uint32_t cbase;      // dynamic part: number of the chunk (dyn_row0, piece 0)
    uint32_t n_real;     // N of the matrix (row stride of Y); == N unless the launch groups rows
};

struct GemmArgs {
    const uint32_t* T;
    float* part;         // fp32 partials: [chunk][2][batch/4][128][4]: slot 0 = the row that ENDS in the chunk, 1 = any other cut row
    uint32_t* ticket;    // per tile row of the launch: contributors that have claimed their turn
    uint32_t* ready;     // per tile row: partials published
    uint32_t* sched;     // [0] next dynamic chunk, [1] CTAs done (the last one resets both)
    uint32_t log2b;
    uint32_t batch;      // columns of the MMA (N): the caller's batch rounded up to a multiple of 16; X rows past the real batch
    uint32_t nreal;      // are zero-filled by TMA (out of bounds of its map) and their Y columns are not stored
    uint32_t nops;
    uint32_t sper;       // static part [0, dyn_base): CTA b starts with its b-th equal share, sper or sper + 1 units
    uint32_t srem;       // ... the first srem shares have sper + 1
    uint32_t dyn_base;   // first unit of the dynamic part (a tile-row boundary)
    uint32_t ndyn;       // chunks of the dynamic part: whole tile rows, or equal pieces of a row that is longer than the cap
    uint32_t total;      // units of the launch
    uint32_t wstages;    // ring of 32 KiB weight tiles (HBM latency: deep)
    uint32_t xstages;    // ring of X tiles [batch x 128] (L2 latency: shallow)
    uint32_t tmem_cols;  // power of two >= 2*batch
    uint32_t early;      // 1: W unchanged since before the preceding kernel -> stream it ahead of griddepcontrol.wait
    uint32_t nacc;       // ROW GROUPS: 1, 2 or 4 tile rows share each X tile.  A unit is then the nacc tiles (nacc*p + rr, tk), rr < nacc, of a
                         // GROUP p of tile rows: the X tile comes out of L2 once instead of nacc times (at batch 128 the X traffic equals
                         // the weight traffic and is worth 12-15 % of the kernel).  ops[].N / units / row_base /
                         // dyn_row0 ... then count GROUPS (the plan ran on N / nacc), ops[].n_real is the matrix's N; nacc accumulators
                         // per segment, double-buffered: 2 * nacc * batch <= 512 TMEM columns.
    GemmOp ops[GM_MAX_OPS];
    alignas(64) CUtensorMap map_x[GM_MAX_OPS];   // X of op j as a 2-D map [batch, K], boxes of [batch x 64]
};

constexpr int GM_THREADS = 224;            // warp 0 scheduler + TMA (W), warp 1 MMA, warp 2 TMA (X), warps 3..6 epilogue
constexpr int GM_MAX_STAGES = 6;
constexpr int GM_QUEUE = 8;                // chunks the scheduler may run ahead of the slowest role
constexpr uint32_t GM_END = 0xffffffffu;

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t c0, uint32_t c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        :: "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// K-major, SWIZZLE_128B shared-memory matrix descriptor (sm_100 format): 8-row atoms of 1024 B.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3FFFF) >> 4) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// Programmatic dependent launch, as in gemv_stream.cu: W (immutable during decode) may be fetched while the stream
// predecessor drains; X, Y, partials and counters wait.  The trigger comes after this grid's own wait.
__device__ __forceinline__ void gm_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void gm_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

// The chunk grid, shared by the kernel and the host (cloak_gemm_plan exposes it to the tests).
// Static part: first unit of share b, and the share that holds unit g.
__host__ __device__ __forceinline__ uint32_t static_begin(const GemmArgs& a, uint32_t b) { return b * a.sper + (b < a.srem ? b : a.srem); }
__host__ __device__ __forceinline__ uint32_t static_chunk_of(const GemmArgs& a, uint32_t g) {
    const uint32_t big = a.srem * (a.sper + 1);
    return g < big ? g / (a.sper + 1) : a.srem + (g - big) / a.sper;
}
// Dynamic part: units [gbeg, gend) of chunk k < a.ndyn -- piece pc of tile row tn of the op whose chunks hold number k.
__host__ __device__ __forceinline__ void dyn_chunk(const GemmArgs& a, uint32_t k, uint32_t& gbeg, uint32_t& gend) {
    uint32_t j = 0;
    while (j + 1 < a.nops && a.ops[j + 1].cbase <= k) ++j;
    const GemmOp& op = a.ops[j];
    const uint32_t loc = k - op.cbase, tn = op.dyn_row0 + loc / op.pieces, pc = loc % op.pieces;
    const uint32_t last = (pc + 1) * op.plen < op.kt ? (pc + 1) * op.plen : op.kt;
    gbeg = op.ubase + tn * op.kt + pc * op.plen;
    gend = op.ubase + tn * op.kt + last;
}

// A launch runs a list of independent ops (cloak_gemm_chain; cloak_gemm is a list of one): the rings, the accumulator
// double buffer and their phases simply continue from chunk to chunk and from op to op, so the weight stream does not
// stop at an op boundary (per-launch head and tail cost ~4 us each; q, k, v, o of a Qwen-32B layer are 13 % of the bytes
// and were 35 % of the time as separate launches).
__global__ void __launch_bounds__(GM_THREADS, 1) gemm_tile128_kernel(const __grid_constant__ CUtensorMap map_w,
                                                                     const __grid_constant__ GemmArgs a) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t wfull[GM_MAX_STAGES], wempty[GM_MAX_STAGES], xfull[GM_MAX_STAGES], xempty[GM_MAX_STAGES],
        tmem_full[2], tmem_empty[2], qfull[GM_QUEUE], qempty[GM_QUEUE];
    __shared__ uint4 queue[GM_QUEUE];                        // {chunk index, first unit, end unit, -}; chunk index GM_END = stop
    __shared__ uint32_t tmem_base_s, last_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // dynamic shared memory is only guaranteed 16-byte aligned: round up to the 1 KiB the 128-byte swizzle needs
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;

    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < GM_MAX_STAGES; ++s) {
            mbar_init(smem_u32(&wfull[s]), 1);
            mbar_init(smem_u32(&wempty[s]), 1);
            mbar_init(smem_u32(&xfull[s]), 1);
            mbar_init(smem_u32(&xempty[s]), 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(smem_u32(&tmem_full[i]), 1);
            mbar_init(smem_u32(&tmem_empty[i]), 4);
        }
        for (int i = 0; i < GM_QUEUE; ++i) {
            mbar_init(smem_u32(&qfull[i]), 1);
            mbar_init(smem_u32(&qempty[i]), 6);              // X producer, MMA issuer, 4 epilogue warps
        }
        fence_barrier_init();
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(&tmem_base_s)), "r"(a.tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;

    const uint32_t xbox = a.batch * 128;                     // bytes of one X box [batch x 64 bf16]
    const uint32_t xtile = 2 * xbox;
    const uint32_t x_base = smem_base + a.wstages * 32768;

    // Every role but the scheduler: next chunk from the queue (false = the launch's sequence is exhausted).
    uint32_t qi = 0;
    auto next_chunk = [&](uint32_t& cidx, uint32_t& gbeg, uint32_t& gend, bool one_lane) -> bool {
        const uint32_t s = qi % GM_QUEUE;
        mbar_wait(smem_u32(&qfull[s]), (qi / GM_QUEUE) & 1);
        const uint4 c = queue[s];
        if (!one_lane) __syncwarp();
        if (one_lane || lane == 0) mbar_arrive(smem_u32(&qempty[s]));
        ++qi;
        cidx = c.x;
        gbeg = c.y;
        gend = c.z;
        return c.x != GM_END;
    };

    if (warp == 0 && lane == 0) {
        // ---------------------------------------------------------------- scheduler + TMA producer, weight tiles (through T)
        if (!a.early) gm_dep_wait();
        uint32_t it = 0, qp = 0;
        auto push = [&](uint32_t cidx, uint32_t gbeg, uint32_t gend) {
            const uint32_t s = qp % GM_QUEUE;
            if (qp >= GM_QUEUE) mbar_wait(smem_u32(&qempty[s]), (qp / GM_QUEUE - 1) & 1);
            queue[s] = make_uint4(cidx, gbeg, gend, 0u);
            mbar_arrive(smem_u32(&qfull[s]));                                        // release: the entry is visible to the waiters
            ++qp;
        };
        auto stream = [&](uint32_t gbeg, uint32_t gend) {
            for (uint32_t j = 0; j < a.nops; ++j) {
                const GemmOp& op = a.ops[j];
                if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;     // this chunk's part of the op, in op units
                const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
                for (uint32_t u = ubeg; u < uend; ++u) {
                    for (uint32_t rr = 0; rr < a.nacc; ++rr, ++it) {
                        const uint32_t s = it % a.wstages, f = it / a.wstages;
                        if (f > 0) mbar_wait(smem_u32(&wempty[s]), (f - 1) & 1);
                        // tile index: tile tk of row nacc * p + rr of the unit's group (nacc == 1: the unit itself)
                        const uint32_t tile = ((u / op.kt) * a.nacc + rr) * op.kt + u % op.kt;
                        const uint64_t off = op.w_offset + (uint64_t)tile * 32768;
                        const uint32_t slot = __ldg(a.T + (off >> a.log2b));
                        const uint64_t byte = ((uint64_t)slot << a.log2b) + (off & ((1ull << a.log2b) - 1));
                        const uint32_t row = (uint32_t)(byte >> 8);                  // pool viewed as rows of 256 B
                        const uint32_t st = smem_base + s * 32768;
                        const uint32_t bar = smem_u32(&wfull[s]);
                        mbar_expect_tx(bar, 32768);
                        tma_load_2d(st, &map_w, 0, row, bar);
                        tma_load_2d(st + 16384, &map_w, 64, row, bar);
                    }
                }
            }
        };
        const uint32_t sbeg = static_begin(a, blockIdx.x), send = static_begin(a, blockIdx.x + 1);
        if (send > sbeg) {                                                           // (a tiny launch has no static part)
            push(blockIdx.x, sbeg, send);
            stream(sbeg, send);
        }
        if (a.early) gm_dep_wait();                                                  // the scheduler's counter is the predecessor's too
        uint32_t k = atomicAdd(a.sched, 1u);
        while (k < a.ndyn) {
            uint32_t gbeg, gend;
            dyn_chunk(a, k, gbeg, gend);
            push(gridDim.x + k, gbeg, gend);
            k = atomicAdd(a.sched, 1u);                                              // in flight while this chunk is issued
            stream(gbeg, gend);
        }
        push(GM_END, GM_END, GM_END);
        __threadfence();
        if (atomicAdd(a.sched + 1, 1u) == gridDim.x - 1) {                           // every CTA has drawn its last chunk: reset
            __threadfence();
            a.sched[0] = 0;
            a.sched[1] = 0;
        }
    } else if (warp == 2 && lane == 0) {
        // ---------------------------------------------------------------- TMA producer, activation tiles (L2-resident)
        gm_dep_wait();
        uint32_t it = 0, cidx, gbeg, gend;
        while (next_chunk(cidx, gbeg, gend, true)) {
            for (uint32_t j = 0; j < a.nops; ++j) {
                const GemmOp& op = a.ops[j];
                if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;
                const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
                for (uint32_t u = ubeg; u < uend; ++u, ++it) {
                    const uint32_t s = it % a.xstages, f = it / a.xstages;
                    if (f > 0) mbar_wait(smem_u32(&xempty[s]), (f - 1) & 1);
                    const uint32_t tk = u % op.kt;
                    const uint32_t st = x_base + s * xtile;
                    const uint32_t bar = smem_u32(&xfull[s]);
                    mbar_expect_tx(bar, xtile);
                    tma_load_2d(st, &a.map_x[j], tk * 128, 0, bar);
                    tma_load_2d(st + xbox, &a.map_x[j], tk * 128 + 64, 0, bar);
                }
            }
        }
    } else if (warp == 1 && lane == 0) {
        // ---------------------------------------------------------------- MMA issuer
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((a.batch >> 3) << 17) | ((128u >> 4) << 24);
        uint32_t it = 0, wit = 0, seg = 0, cidx, gbeg, gend;                    // it (X ring), wit (W ring), seg run on across chunks and ops
        const uint32_t nacc = a.nacc;                                           // accumulators per segment
        auto acquire_acc = [&]() {                                              // accumulator seg & 1 drained by the epilogue?
            if (seg >= 2) {
                mbar_wait(smem_u32(&tmem_empty[seg & 1]), ((seg >> 1) - 1) & 1);
                tc_fence_after();
            }
        };
        while (next_chunk(cidx, gbeg, gend, true)) {
            for (uint32_t j = 0; j < a.nops; ++j) {
                const GemmOp& op = a.ops[j];
                if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;
                const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
                uint32_t cur_tn = ubeg / op.kt;
                bool first = true;
                acquire_acc();
                for (uint32_t u = ubeg; u < uend; ++u, ++it) {
                    const uint32_t tn = u / op.kt;
                    if (tn != cur_tn) {
                        tc_commit(smem_u32(&tmem_full[seg & 1]));                // accumulator of the finished tile row
                        ++seg;
                        cur_tn = tn;
                        first = true;
                        acquire_acc();
                    }
                    const uint32_t xs = it % a.xstages;
                    mbar_wait(smem_u32(&xfull[xs]), (it / a.xstages) & 1);
                    const uint32_t sx = x_base + xs * xtile;
                    for (uint32_t rr = 0; rr < nacc; ++rr, ++wit) {              // the group's weight tiles against one X tile
                        const uint32_t ws = wit % a.wstages;
                        mbar_wait(smem_u32(&wfull[ws]), (wit / a.wstages) & 1);
                        tc_fence_after();
                        const uint32_t st = smem_base + ws * 32768;
                        const uint32_t d = tmem_base + ((seg & 1) * nacc + rr) * a.batch;
#pragma unroll
                        for (int box = 0; box < 2; ++box) {
                            const uint64_t ad = umma_desc_sw128(st + box * 16384);
                            const uint64_t bd = umma_desc_sw128(sx + box * xbox);
#pragma unroll
                            for (int k = 0; k < 4; ++k)                          // UMMA_K = 16 bf16 = 32 B inside the atom
                                tc_mma_bf16(d, ad + 2 * k, bd + 2 * k, idesc, (first && box == 0 && k == 0) ? 0u : 1u);
                        }
                        tc_commit(smem_u32(&wempty[ws]));                        // frees the stage when its MMAs retire
                    }
                    first = false;
                    tc_commit(smem_u32(&xempty[xs]));
                }
                tc_commit(smem_u32(&tmem_full[seg & 1]));
                ++seg;
            }
        }
    } else if (warp >= 3) {
        // ---------------------------------------------------------------- epilogue (4 warps = 4 TMEM lane quarters)
        const uint32_t q = warp & 3, r = q * 32 + lane;
        const int etid = threadIdx.x - 96;
        gm_dep_wait();
        if (etid == 0) gm_dep_launch();
        const uint32_t nout = a.batch * 128;
        uint32_t seg = 0, cidx, gbeg, gend;
        while (next_chunk(cidx, gbeg, gend, false)) {
            for (uint32_t j = 0; j < a.nops; ++j) {
                const GemmOp& op = a.ops[j];
                if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;
                const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
                const uint32_t kt = op.kt;
                for (uint32_t u = ubeg; u < uend; ++seg) {
                    const uint32_t tn = u / kt;
                    const uint32_t t_first = tn * kt, t_last = t_first + kt - 1;
                    const uint32_t seg_last = min(uend - 1, t_last);
                    // the chunks that meet this tile row, in sequence order: its contributors
                    uint32_t c_first, ncontrib;
                    if (tn >= op.dyn_row0) {                                     // dynamic part: the row's pieces
                        c_first = gridDim.x + op.cbase + (tn - op.dyn_row0) * op.pieces;
                        ncontrib = op.pieces;
                    } else {
                        c_first = static_chunk_of(a, op.ubase + t_first);
                        ncontrib = static_chunk_of(a, op.ubase + t_last) - c_first + 1;
                    }
                    const uint32_t me = cidx - c_first;
                    const bool complete = ncontrib == 1;
                    // one accumulator per tile row of the group: rows nacc * tn + rr, same contributors, own tickets
                    for (uint32_t rr = 0; rr < a.nacc; ++rr) {
                    const uint32_t tnr = a.nacc * tn + rr;
                    const uint32_t row = (op.row_base + tn) * a.nacc + rr;
                    bool last = false;
                    if (!complete) {
                        // Tickets: whoever draws the last one finishes the row.  With the static chunks that is the row's
                        // first contributor (it meets the row at the END of its chunk, the next one at the start of its own);
                        // in the dynamic part it is whoever comes last.
                        if (etid == 0) last_s = (atomicAdd(a.ticket + row, 1u) == ncontrib - 1) ? 1u : 0u;
                        epi_bar();
                        last = last_s != 0;
                    }
                    if (rr == 0) mbar_wait(smem_u32(&tmem_full[seg & 1]), (seg >> 1) & 1);
                    tc_fence_after();
                    const uint32_t taddr = tmem_base + ((q * 32) << 16) + ((seg & 1) * a.nacc + rr) * a.batch;
                    const size_t n = (size_t)tnr * 128 + r;
                    if (last) {
                        if (etid == 0) {
                            uint32_t seen;
                            do {
                                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(a.ready + row) : "memory");
                                if (seen != ncontrib - 1) __nanosleep(64);
                            } while (seen != ncontrib - 1);
                            a.ticket[row] = 0;                                   // self-reset for the next launch
                            a.ready[row] = 0;
                        }
                        epi_bar();
                        __threadfence();
                    }
                    // partial of contributor p of this row: slot 0 of its chunk if the row ENDS there, else slot 1; a slot is
                    // [batch/4][128 rows][4] fp32, so that a thread moves its row's values of 4 batch columns as one float4
                    auto slot_of = [&](uint32_t p) {
                        return reinterpret_cast<float4*>(a.part + (((size_t)(c_first + p) * 2 + (p == ncontrib - 1 ? 0 : 1)) * a.nacc + rr) * nout) + r;
                    };
                    float4* mine = slot_of(me);
                    for (uint32_t c = 0; c < a.batch; c += 32) {                 // 32 batch columns per round (16 in a last odd one)
                        const bool two = c + 16 < a.batch;
                        uint32_t v0[16], v1[16];
                        tc_ld16(taddr + c, v0);
                        if (two) tc_ld16(taddr + c + 16, v1);
                        if (last) {
                            // own part from TMEM, the others' from L2, added in chunk order; 2 x 8 float4 loads in flight per thread
                            float sum[32];
#pragma unroll
                            for (int i = 0; i < 32; ++i) sum[i] = 0.f;
                            for (uint32_t p = 0; p < ncontrib; p += 2) {
                                float4 x[2][8];
#pragma unroll
                                for (int pp = 0; pp < 2; ++pp) {
                                    const bool ld = p + pp < ncontrib && p + pp != me;
                                    const float4* src = slot_of(ld ? p + pp : 0) + (size_t)(c / 4) * 128;
#pragma unroll
                                    for (int i = 0; i < 8; ++i)
                                        x[pp][i] = (ld && (i < 4 || two)) ? __ldcg(src + i * 128) : make_float4(0.f, 0.f, 0.f, 0.f);
                                }
#pragma unroll
                                for (int pp = 0; pp < 2; ++pp) {
                                    if (p + pp == me) {
#pragma unroll
                                        for (int i = 0; i < 16; ++i) {
                                            sum[i] += __uint_as_float(v0[i]);
                                            if (two) sum[16 + i] += __uint_as_float(v1[i]);
                                        }
                                    } else if (p + pp < ncontrib) {
#pragma unroll
                                        for (int i = 0; i < 8; ++i) {
                                            sum[4 * i] += x[pp][i].x;
                                            sum[4 * i + 1] += x[pp][i].y;
                                            sum[4 * i + 2] += x[pp][i].z;
                                            sum[4 * i + 3] += x[pp][i].w;
                                        }
                                    }
                                }
                            }
#pragma unroll
                            for (int i = 0; i < 32; ++i)
                                if (c + i < a.nreal) op.y[(size_t)(c + i) * op.n_real + n] = __float2bfloat16_rn(sum[i]);
                        } else if (complete) {
#pragma unroll
                            for (int i = 0; i < 16; ++i) {
                                if (c + i < a.nreal) op.y[(size_t)(c + i) * op.n_real + n] = __float2bfloat16_rn(__uint_as_float(v0[i]));
                                if (c + 16 + i < a.nreal) op.y[(size_t)(c + 16 + i) * op.n_real + n] = __float2bfloat16_rn(__uint_as_float(v1[i]));
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                __stcg(mine + (size_t)(c / 4 + i) * 128, make_float4(__uint_as_float(v0[4 * i]), __uint_as_float(v0[4 * i + 1]),
                                                                                     __uint_as_float(v0[4 * i + 2]), __uint_as_float(v0[4 * i + 3])));
                                if (two)
                                    __stcg(mine + (size_t)(c / 4 + 4 + i) * 128, make_float4(__uint_as_float(v1[4 * i]), __uint_as_float(v1[4 * i + 1]),
                                                                                             __uint_as_float(v1[4 * i + 2]), __uint_as_float(v1[4 * i + 3])));
                            }
                        }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0 && rr + 1 == a.nacc) mbar_arrive(smem_u32(&tmem_empty[seg & 1]));    // all accumulators drained
                    if (!complete && !last) {                                    // publish this chunk's part of the cut row
                        __threadfence();
                        epi_bar();
                        if (etid == 0) asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(a.ready + row), "r"(1u) : "memory");
                    }
                    }
                    u = seg_last + 1;
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(a.tmem_cols) : "memory");
    }
}

static cloak_status make_map(CUtensorMap* map, const void* base, uint64_t inner, uint64_t rows, uint64_t pitch_bytes,
                             uint32_t box_inner, uint32_t box_rows) {
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    cuuint64_t dims[2] = {inner, rows};
    cuuint64_t strides[1] = {pitch_bytes};
    cuuint32_t box[2] = {box_inner, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CLOAK_CU(d->TensorMapEncodeTiled(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box,
                                     estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE));
    return CLOAK_OK;
}

extern std::atomic<bool> g_gemv_pdl;      // gemv_stream.cu: the PDL A/B switch (cloak_set_gemv_engine(2) turns it off)
cloak_status check_linear(const cloak_pool* pool, const cloak_tensor* w, const void* x, void* y, const char* who);

static cloak_status gemm_check(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y, uint32_t batch,
                               const char* who) {
    cloak_status st = check_linear(pool, w, d_x, d_y, who);
    if (st != CLOAK_OK) return st;
    if (batch < 1 || batch > 256) return fail(CLOAK_ERR_INVALID, "%s: batch must be in 1..256", who);
    if (w->dt != CLOAK_BF16 || w->layout != CLOAK_TILE128) return fail(CLOAK_ERR_UNSUPPORTED, "%s: needs CLOAK_BF16 in CLOAK_TILE128 layout", who);
    if (w->N % 128 || w->K % 128) return fail(CLOAK_ERR_ALIGN, "%s: N and K must be multiples of 128", who);
    if (pool->block < 32768) return fail(CLOAK_ERR_UNSUPPORTED, "%s: block_bytes must be >= 32 KiB (one 128x128 bf16 tile)", who);
    return CLOAK_OK;
}

// Schedule knobs (cloak_set_gemm_schedule): percentage of the launch's tiles that is dealt out statically, and the cap on
// the tiles of a dynamic chunk (0 = by batch).
static std::atomic<int> g_static_pct{75};
static std::atomic<int> g_dchunk{0};

constexpr uint32_t GM_MAX_ROWS = 100000;   // tile rows per launch: two counters each in the pool's counter scratch
static std::atomic<int> g_gemm_engine{0};  // cloak_set_gemm_engine: 0 = pairs of tile rows where they still fill the SMs, 1 = never, 2 = fours / 3 = pairs wherever N allows
// Measured (16 Qwen-32B-shaped layers, >= 1 s loops, of the measured copy peak): single rows 0.912 / 0.827 / 0.713 at batch 32 / 64 /
// 128; pairs 0.987 / 0.910 / 0.799; fours (batch <= 64) 0.926 / 0.855 -- a group of four quarters the dynamic chunk and doubles
// the rows a chunk boundary cuts, which costs more than the second halving of the X traffic returns.
// Tile rows per group for an MMA batch (2 * nacc * batch <= 512 TMEM columns) and a list of matrices (N a multiple of 128 * nacc).
// A chunk boundary cuts nacc tile rows instead of one (nacc fp32 partials and as many reductions), so a group pays only in a
// launch that gives every CTA a long share: measured on Qwen-32B-shaped projections, pairs lose below ~150 tiles per CTA
// (one projection: gate 50 -> 56 us at batch 32, 60 -> 80 us at batch 128) and win above ~175 (a layer's MLP or more).
// Nor may the grouped units stop filling the SMs under gemm_plan's cap on chunks per row.
constexpr uint64_t GM_GROUP_MIN_TILES_PER_CTA = 160;
static uint32_t gemm_plan_ctas(uint64_t total, uint32_t max_kt, uint32_t batch, int sms) {
    uint32_t cap = 512 / batch;
    cap = cap < 4 ? 4 : (cap > 10 ? 10 : cap);
    const uint32_t minper = (max_kt + cap - 1) / cap;
    const uint64_t c = total / minper;
    return (uint32_t)(c < 1 ? 1 : (c > (uint64_t)sms ? (uint64_t)sms : c));
}
template <typename GetN, typename GetK>
static uint32_t gemm_grouping(uint32_t mma_batch, uint32_t n, int sms, GetN N, GetK K) {
    const int eng = g_gemm_engine.load(std::memory_order_relaxed);
    uint32_t nacc = eng == 1 ? 1u : (mma_batch <= 64 && eng == 2 ? 4u : (mma_batch <= 128 ? 2u : 1u));
    if (mma_batch < 32 && eng == 0) nacc = 1;       // (below that the X tile is a small fraction of the weight tile)
    uint64_t tiles = 0;
    uint32_t max_kt = 0;
    for (uint32_t j = 0; j < n; ++j) {
        while (nacc > 1 && N(j) % (128 * nacc)) nacc /= 2;
        tiles += (uint64_t)(N(j) / 128) * (K(j) / 128);
        if (K(j) / 128 > max_kt) max_kt = K(j) / 128;
    }
    if (eng == 0 && tiles < GM_GROUP_MIN_TILES_PER_CTA * (uint64_t)sms) nacc = 1;
    while (eng == 0 && nacc > 1 && gemm_plan_ctas(tiles / nacc, max_kt, mma_batch, sms) < gemm_plan_ctas(2 * tiles / nacc, max_kt, mma_batch, sms)) nacc /= 2;
    return nacc;
}

// The chunk grid of one launch: fills the schedule fields of a (ops[j].N/kt/units/ubase/row_base/dyn_row0/pieces/plen/cbase,
// sper, srem, dyn_base, ndyn, total, nops) from the shapes alone.  `batch` is the MMA's N (a multiple of 16).
// The launch's tiles -- all ops back to back, each tn-major -- form one sequence.  Its first g_static_pct percent, up to a
// tile-row boundary, are the static part: CTA b takes the b-th equal share of it.  The rows after that are the dynamic
// part: whole tile rows (no split-K at all), or equal pieces of a row that is longer than the cap, drawn from a counter
// as the CTAs become free.  Every piece boundary costs one partial [batch x 128] fp32 and a share of a reduction, so the
// cap grows with the batch.
// nacc: the launch groups tile rows -- N[] are then the matrices' N / nacc, a unit is nacc tiles and a dynamic chunk holds 1 / nacc as many.
static cloak_status gemm_plan(GemmArgs& a, const uint32_t* N, const uint32_t* K, uint32_t n, uint32_t batch, int sms,
                              uint32_t* ctas_out, uint64_t* rows_out, uint32_t nacc = 1) {
    uint64_t rows = 0, total = 0;
    uint32_t max_kt = 0;
    a.nops = n;
    for (uint32_t j = 0; j < n; ++j) {
        GemmOp& o = a.ops[j];
        o.N = N[j];
        o.kt = K[j] / 128;
        if (o.kt > max_kt) max_kt = o.kt;
        const uint64_t units64 = (uint64_t)(N[j] / 128) * o.kt;
        if (total + units64 > 0x7fffffffull) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: too many tiles in one launch");
        o.units = (uint32_t)units64;
        o.ubase = (uint32_t)total;
        o.row_base = (uint32_t)rows;
        o.n_real = nacc * N[j];
        total += units64;
        rows += N[j] / 128;
    }
    if (rows > GM_MAX_ROWS) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: too many output rows for the tile counters");
    // At most ~cap chunks per tile row (the fp32 partials are batch * 512 B each): small launches use fewer CTAs.
    uint32_t cap = 512 / batch;
    cap = cap < 4 ? 4 : (cap > 10 ? 10 : cap);
    const uint32_t minper = (max_kt + cap - 1) / cap;
    const uint32_t ctas = gemm_plan_ctas(total, max_kt, batch, sms);
    const int dchunk = g_dchunk.load(std::memory_order_relaxed), static_pct = g_static_pct.load(std::memory_order_relaxed);
    uint32_t dmax = dchunk > 0 ? (uint32_t)dchunk : (batch >= 128 ? 40u : 20u);
    if (dchunk == 0) dmax /= nacc;
    if (dmax < minper) dmax = minper;
    // A launch with less than a few dynamic chunks' worth of tiles per CTA is dealt out statically: its tail would be as
    // long as a chunk, and there is little to balance.
    const uint64_t target = (total / ctas < 4ull * dmax && dchunk == 0) ? total : total * (uint64_t)static_pct / 100;
    uint32_t ndyn = 0;
    a.dyn_base = (uint32_t)total;
    for (uint32_t j = 0; j < n; ++j) {
        GemmOp& o = a.ops[j];
        const uint32_t tile_rows = o.N / 128;
        if (o.ubase + (uint64_t)o.units <= target) o.dyn_row0 = tile_rows;                 // wholly static
        else if (o.ubase >= target) o.dyn_row0 = 0;                                         // wholly dynamic
        else o.dyn_row0 = (uint32_t)((target - o.ubase) / o.kt);                            // the boundary row: rounded down
        if (o.dyn_row0 < tile_rows && a.dyn_base == (uint32_t)total) a.dyn_base = o.ubase + o.dyn_row0 * o.kt;
        o.pieces = (o.kt + dmax - 1) / dmax;
        o.plen = (o.kt + o.pieces - 1) / o.pieces;
        o.pieces = (o.kt + o.plen - 1) / o.plen;                                            // no empty last piece
        o.cbase = ndyn;
        ndyn += (tile_rows - o.dyn_row0) * o.pieces;
    }
    a.sper = a.dyn_base / ctas;
    a.srem = a.dyn_base % ctas;
    a.ndyn = ndyn;
    a.total = (uint32_t)total;
    *ctas_out = ctas;
    *rows_out = rows;
    return CLOAK_OK;
}

// One launch of n <= GM_MAX_OPS checked ops.
static cloak_status gemm_launch(const cloak_pool* pool, const cloak_gemm_op* ops, uint32_t n, uint32_t batch, cudaStream_t s) {
    cloak_status st;
    if (!pool->tmap_ready) {
        cloak_pool* p = const_cast<cloak_pool*>(pool);
        // (real pages: both halves of the pool's virtual range, see cloak_pool::page_half; unmapped parts are never addressed)
        st = make_map(&p->tmap_tile128, pool->base, 128, (pool->vmm ? 2 : 1) * (pool->bytes() / 256), 256, 64, 128);
        if (st != CLOAK_OK) return st;
        p->tmap_ready = true;
    }
    GemmArgs a;
    a.T = pool->d_T;
    a.log2b = pool->log2_block;
    const uint32_t nreal = batch;
    batch = (batch + 15) & ~15u;         // the MMA's N; TMA zero-fills the X rows past the real batch
    a.batch = batch;
    a.nreal = nreal;
    const int sms = sm_count(pool->device);
    uint32_t Ns[GM_MAX_OPS], Ks[GM_MAX_OPS], ctas = 0;
    uint64_t rows = 0;
    // Row groups (GemmArgs::nacc): as many tile rows per X tile as the 512 TMEM columns hold accumulators for, if every matrix
    // of the launch has a multiple of that many tile rows.
    const uint32_t nacc = gemm_grouping(batch, n, sms, [&](uint32_t j) { return ops[j].w.N; }, [&](uint32_t j) { return ops[j].w.K; });
    a.nacc = nacc;
    for (uint32_t j = 0; j < n; ++j) {
        const cloak_tensor& w = ops[j].w;
        Ns[j] = w.N / nacc;
        Ks[j] = w.K;
        st = make_map(&a.map_x[j], ops[j].d_x, w.K, nreal, (uint64_t)w.K * 2, 64, batch);
        if (st != CLOAK_OK) return st;
        a.ops[j].w_offset = w.w_offset;
        a.ops[j].y = static_cast<__nv_bfloat16*>(ops[j].d_y);
    }
    st = gemm_plan(a, Ns, Ks, n, batch, sms, &ctas, &rows, nacc);
    if (st != CLOAK_OK) return st;
    rows *= nacc;                                    // ticket / ready counters: one per real tile row
    if ((2 * rows + 2) * 4 > WS_COUNTER_BYTES) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: too many output rows for the tile counters");
    const uint64_t nchunks = (uint64_t)ctas + a.ndyn;
    const uint64_t part_bytes = nchunks * 2 * nacc * batch * 128 * 4;
    const uint32_t xtile = batch * 256;
    a.xstages = 2;
    uint32_t wst = (224u * 1024u - a.xstages * xtile) / 32768u;
    if (wst > GM_MAX_STAGES) wst = GM_MAX_STAGES;
    if (wst < 2) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: batch too large for the shared-memory ring");
    a.wstages = wst;
    a.tmem_cols = 32;
    while (a.tmem_cols < 2 * nacc * batch) a.tmem_cols <<= 1;
    st = pool_workspace(pool, WS_COUNTER_BYTES + part_bytes, s);
    if (st != CLOAK_OK) return st;
    a.ticket = reinterpret_cast<uint32_t*>(pool->ws);
    a.ready = a.ticket + rows;
    a.sched = a.ready + rows;
    a.part = reinterpret_cast<float*>(pool->ws + WS_COUNTER_BYTES);

    const size_t smem = (size_t)a.wstages * 32768 + (size_t)a.xstages * xtile + 1024;
    static std::atomic<uint64_t> opted{0};
    st = smem_opt_in(gemm_tile128_kernel, 226 * 1024, pool->device, opted);
    if (st != CLOAK_OK) return st;
    const bool pdl = g_gemv_pdl.load(std::memory_order_relaxed);
    a.early = (pdl && !pool->dirty) ? 1u : 0u;
    if (pool->dirty && pool->dirty_stream == s) pool->dirty = false;   // this launch waits for the writer in full
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ctas);
    cfg.blockDim = dim3(GM_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    CLOAK_CUDA(cudaLaunchKernelEx(&cfg, gemm_tile128_kernel, pool->tmap_tile128, a));
    launched();
    return CLOAK_OK;
}

}  // namespace cloak

using namespace cloak;

extern "C" cloak_status cloak_set_gemm_schedule(int static_pct, int dyn_chunk_tiles) {
    if (static_pct < 0 || static_pct > 100 || dyn_chunk_tiles < 0 || dyn_chunk_tiles > 4096)
        return fail(CLOAK_ERR_INVALID, "set_gemm_schedule: static_pct in 0..100, dyn_chunk_tiles in 0..4096");
    g_static_pct.store(static_pct);
    g_dchunk.store(dyn_chunk_tiles);
    return CLOAK_OK;
}

extern "C" cloak_status cloak_set_gemm_engine(int engine) {
    if (engine < 0 || engine > 3) return fail(CLOAK_ERR_INVALID, "set_gemm_engine: 0 (automatic: pairs of tile rows), 1 (never), 2 (fours wherever N and TMEM allow) or 3 (pairs wherever N allows)");
    g_gemm_engine.store(engine);
    return CLOAK_OK;
}

extern "C" cloak_status cloak_gemm_plan(uint32_t n_ops, const uint32_t* h_N, const uint32_t* h_K, uint32_t batch, uint32_t sms,
                                        uint32_t max_chunks, uint32_t* h_begin, uint32_t* h_end, uint32_t* h_nchunks,
                                        uint32_t* h_nstatic, uint32_t* h_group) {
    if (!h_N || !h_K || !h_nchunks || !h_nstatic || !h_group || n_ops == 0 || n_ops > (uint32_t)GM_MAX_OPS)
        return fail(CLOAK_ERR_INVALID, "gemm_plan: 1..%d ops", GM_MAX_OPS);
    if (batch < 1 || batch > 256 || sms < 1) return fail(CLOAK_ERR_INVALID, "gemm_plan: batch in 1..256, sms >= 1");
    for (uint32_t j = 0; j < n_ops; ++j)
        if (h_N[j] == 0 || h_K[j] == 0 || h_N[j] % 128 || h_K[j] % 128) return fail(CLOAK_ERR_ALIGN, "gemm_plan: N and K must be multiples of 128");
    GemmArgs a;
    uint32_t ctas = 0;
    uint64_t rows = 0;
    const uint32_t cols = (batch + 15) & ~15u;
    const uint32_t nacc = gemm_grouping(cols, n_ops, (int)sms, [&](uint32_t j) { return h_N[j]; }, [&](uint32_t j) { return h_K[j]; });
    uint32_t Ng[GM_MAX_OPS];
    for (uint32_t j = 0; j < n_ops; ++j) Ng[j] = h_N[j] / nacc;
    cloak_status st = gemm_plan(a, Ng, h_K, n_ops, cols, (int)sms, &ctas, &rows, nacc);
    if (st != CLOAK_OK) return st;
    *h_group = nacc;
    *h_nstatic = ctas;
    *h_nchunks = ctas + a.ndyn;
    if (!h_begin || !h_end) return CLOAK_OK;
    if (max_chunks < ctas + a.ndyn) return fail(CLOAK_ERR_INVALID, "gemm_plan: %u chunks, room for %u", ctas + a.ndyn, max_chunks);
    for (uint32_t b = 0; b < ctas; ++b) {                // the same functions the kernel calls
        h_begin[b] = static_begin(a, b);
        h_end[b] = static_begin(a, b + 1);
    }
    for (uint32_t k = 0; k < a.ndyn; ++k) dyn_chunk(a, k, h_begin[ctas + k], h_end[ctas + k]);
    return CLOAK_OK;
}

extern "C" cloak_status cloak_gemm(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                                   uint32_t batch, void* stream) {
    cloak_status st = gemm_check(pool, w, d_x, d_y, batch, "gemm");
    if (st != CLOAK_OK) return st;
    DeviceGuard g(pool->device);
    cloak_gemm_op op;
    op.w = *w;
    op.d_x = d_x;
    op.d_y = d_y;
    return gemm_launch(pool, &op, 1, batch, (cudaStream_t)stream);
}

extern "C" cloak_status cloak_gemm_chain_scratch_bytes(const cloak_pool* pool, const cloak_gemm_op* h_ops, uint32_t n_ops,
                                                       uint32_t batch, uint64_t* h_bytes) {
    if (!h_ops || n_ops == 0 || !h_bytes) return fail(CLOAK_ERR_INVALID, "gemm_chain_scratch_bytes: NULL argument or no ops");
    for (uint32_t i = 0; i < n_ops; ++i) {
        cloak_status st = gemm_check(pool, &h_ops[i].w, h_ops[i].d_x, h_ops[i].d_y, batch, "gemm_chain_scratch_bytes");
        if (st != CLOAK_OK) return st;
    }
    const int sms = sm_count(pool->device);
    const uint32_t cols = (batch + 15) & ~15u;
    uint64_t need = 0;
    for (uint32_t i = 0; i < n_ops;) {                      // the same split into launches as cloak_gemm_chain
        uint32_t n = 0, Ns[GM_MAX_OPS], Ks[GM_MAX_OPS];
        uint64_t rows = 0;
        while (i + n < n_ops && n < (uint32_t)GM_MAX_OPS && rows + h_ops[i + n].w.N / 128 <= GM_MAX_ROWS) {
            Ns[n] = h_ops[i + n].w.N;
            Ks[n] = h_ops[i + n].w.K;
            rows += h_ops[i + n++].w.N / 128;
        }
        if (n == 0) return fail(CLOAK_ERR_UNSUPPORTED, "gemm_chain_scratch_bytes: op %u has too many output rows", i);
        GemmArgs a;
        uint32_t ctas = 0;
        const uint32_t nacc = gemm_grouping(cols, n, sms, [&](uint32_t j) { return Ns[j]; }, [&](uint32_t j) { return Ks[j]; });
        for (uint32_t j = 0; j < n; ++j) Ns[j] /= nacc;
        cloak_status st = gemm_plan(a, Ns, Ks, n, cols, sms, &ctas, &rows, nacc);
        if (st != CLOAK_OK) return st;
        const uint64_t b = WS_COUNTER_BYTES + ((uint64_t)ctas + a.ndyn) * 2 * nacc * cols * 128 * 4;
        if (b > need) need = b;
        i += n;
    }
    *h_bytes = need;
    return CLOAK_OK;
}

extern "C" cloak_status cloak_gemm_chain(const cloak_pool* pool, const cloak_gemm_op* h_ops, uint32_t n_ops, uint32_t batch,
                                         void* stream) {
    if (!h_ops || n_ops == 0) return fail(CLOAK_ERR_INVALID, "gemm_chain: no ops");
    for (uint32_t i = 0; i < n_ops; ++i) {
        cloak_status st = gemm_check(pool, &h_ops[i].w, h_ops[i].d_x, h_ops[i].d_y, batch, "gemm_chain");
        if (st != CLOAK_OK) return st;
    }
    DeviceGuard g(pool->device);
    for (uint32_t i = 0; i < n_ops;) {                      // at most GM_MAX_OPS ops and GM_MAX_ROWS tile rows per launch
        uint32_t n = 0;
        uint64_t rows = 0;
        while (i + n < n_ops && n < (uint32_t)GM_MAX_OPS && rows + h_ops[i + n].w.N / 128 <= GM_MAX_ROWS) rows += h_ops[i + n++].w.N / 128;
        if (n == 0) return fail(CLOAK_ERR_UNSUPPORTED, "gemm_chain: op %u has too many output rows", i);
        cloak_status st = gemm_launch(pool, h_ops + i, n, batch, (cudaStream_t)stream);
        if (st != CLOAK_OK) return st;
        i += n;
    }
    return CLOAK_OK;
}
