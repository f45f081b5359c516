// S7 cloak_gemm: batch 16..256 contraction on tcgen05 tensor cores, W tiles fetched by TMA through the table.
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
//   * Units = tiles, numbered tn-major (= TILE128 storage order), the ops of a launch back to back, cut into equal
//     contiguous ranges, one per persistent CTA (stream-K over the whole op list): HBM-bound (AI = batch flop/B < ridge), so what matters is that every SM
//     streams the same bytes with a full TMA ring.  Roles: warp 0 TMA producer, warp 1 MMA issuer (one lane)
//     + TMEM allocator, warp 2 TMA producer for X (own shallow ring), warps 3-6 epilogue (tcgen05.ld 32x32b, one TMEM lane quarter each).
//   * A tile row wholly inside a CTA's range is stored as bf16 straight from TMEM; one cut by a range boundary
//     has its later contributors write fp32 partials; the row's first contributor adds them, in contributor order, to
//     its own accumulator as it drains it (deterministic; identical for cloaked and identity-table pools).
//   * PAIR variant (batch >= 64 by default): the grid is launched as clusters of two CTAs (one TPC) that work as a
//     `cta_group::2` pair on TWO adjacent tile rows with the same k tile: each CTA streams its own W tile and only HALF
//     of the X tile (batch/2 rows), the leader issues one M = 256 MMA that reads B from both CTAs' shared memory, and
//     each CTA drains its own 128 TMEM lanes.  Units are then (tile-row pair, k tile), one range per pair.  At batch
//     128 the X tile is as large as the W tile, so this takes the L2 -> SM traffic from 2 x W to 1.5 x W.
#include <cuda_bf16.h>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

constexpr int GM_MAX_OPS = 16;             // ops per launch (one X tensor map of 128 B each in the kernel parameters)

struct GemmOp {
    uint64_t w_offset;
    __nv_bfloat16* y;
    uint64_t part_base;  // float offset of this op's partials: [tile row][maxc][batch][128]
    uint32_t N;
    uint32_t kt;         // k tiles per tile row = K/128
    uint32_t units;      // (N/128) * kt; pair variant: ceil(N/256) * kt
    uint32_t ubase;      // this op's first unit in the launch's unit sequence (ops back to back)
    uint32_t maxc;       // max contributors per tile row
    uint32_t row_base;   // index of this op's first tile-row counter
};

struct GemmArgs {
    const uint32_t* T;
    float* part;
    uint32_t* counters;
    uint32_t log2b;
    uint32_t batch;
    uint32_t nops;
    uint32_t per;        // units per range: the launch's units (all ops back to back) are cut into equal contiguous ranges
    uint32_t total;      // units of the launch
    uint32_t wstages;    // ring of 32 KiB weight tiles (HBM latency: deep)
    uint32_t xstages;    // ring of X tiles [batch x 128] (L2 latency: shallow)
    uint32_t tmem_cols;  // power of two >= 2*batch
    uint32_t early;      // 1: W unchanged since before the preceding kernel -> stream it ahead of griddepcontrol.wait
    GemmOp ops[GM_MAX_OPS];
    alignas(64) CUtensorMap map_x[GM_MAX_OPS];   // X of op j as a 2-D map [batch, K], boxes of [batch x 64]
};

constexpr int GM_THREADS = 224;            // warp 0 TMA (W), warp 1 MMA, warp 2 TMA (X), warps 3..6 epilogue
constexpr int GM_MAX_STAGES = 6;

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t c0, uint32_t c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
// cta_group::2 flavour: executed by both CTAs of the pair, the data lands in the issuing CTA's shared memory, the bytes
// are counted on the LEADER's barrier (`bar` is a shared::cluster address).
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, uint32_t c0, uint32_t c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_bar) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" :: "r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
// Pair flavours: the arrival goes to the barrier at this offset in BOTH CTAs; the MMA spans both CTAs' tensor cores.
__device__ __forceinline__ void tc_commit_pair(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 :: "r"(bar), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void tc_mma_bf16_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        :: "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
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

// A launch runs a list of independent ops (cloak_gemm_chain; cloak_gemm is a list of one): every role walks the list,
// the rings, the accumulator double buffer and their phases simply continue from op to op, so the weight stream does not
// stop at an op boundary (per-launch head and tail cost ~4 us each; q, k, v, o of a Qwen-32B layer are 13 % of the bytes
// and were 35 % of the time as separate launches).
template <bool PAIR>
__global__ void __launch_bounds__(GM_THREADS, 1) gemm_tile128_kernel(const __grid_constant__ CUtensorMap map_w,
                                                                     const __grid_constant__ GemmArgs a) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t wfull[GM_MAX_STAGES], wempty[GM_MAX_STAGES], xfull[GM_MAX_STAGES], xempty[GM_MAX_STAGES],
        tmem_full[2], tmem_empty[2];
    __shared__ uint32_t tmem_base_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // dynamic shared memory is only guaranteed 16-byte aligned: round up to the 1 KiB the 128-byte swizzle needs
    // (same offset in both CTAs of a pair: same kernel, same static shared memory)
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t crank = PAIR ? cluster_ctarank() : 0u;             // 0 = leader (issues the MMAs, owns the full barriers)
    const uint32_t rank_in_grid = PAIR ? blockIdx.x / 2 : blockIdx.x;  // one range per CTA, or per CTA pair
    const uint32_t gbeg = rank_in_grid * a.per, gend = min(gbeg + a.per, a.total);

    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < GM_MAX_STAGES; ++s) {
            mbar_init(smem_u32(&wfull[s]), 1);
            mbar_init(smem_u32(&wempty[s]), 1);
            mbar_init(smem_u32(&xfull[s]), 1);
            mbar_init(smem_u32(&xempty[s]), 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(smem_u32(&tmem_full[i]), 1);
            mbar_init(smem_u32(&tmem_empty[i]), PAIR ? 8 : 4);        // the epilogue warps of both CTAs arrive at the leader's
        }
        fence_barrier_init();
    }
    if (warp == 1) {
        if (PAIR) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;"
                         :: "r"(smem_u32(&tmem_base_s)), "r"(a.tmem_cols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                         :: "r"(smem_u32(&tmem_base_s)), "r"(a.tmem_cols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    tc_fence_before();
    __syncthreads();
    if (PAIR) cluster_sync_all();                                     // the peer's barriers are initialised before anything lands
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;

    const uint32_t xbox = (PAIR ? a.batch / 2 : a.batch) * 128;      // bytes of this CTA's X box [rows x 64 bf16]
    const uint32_t xtile = 2 * xbox;
    const uint32_t x_base = smem_base + a.wstages * 32768;

    if (warp == 0 && lane == 0) {
        // ---------------------------------------------------------------- TMA producer, weight tiles (through T)
        if (!a.early) gm_dep_wait();
        uint32_t it = 0;
        for (uint32_t j = 0; j < a.nops; ++j) {
            const GemmOp& op = a.ops[j];
            if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;         // this range's part of the op, in op units
            const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
            const uint32_t tile_rows = op.N / 128;
            for (uint32_t u = ubeg; u < uend; ++u, ++it) {
                const uint32_t s = it % a.wstages, f = it / a.wstages;
                if (f > 0) mbar_wait(smem_u32(&wempty[s]), (f - 1) & 1);
                uint32_t tile = u, bar = smem_u32(&wfull[s]);
                bool valid = true;
                if (PAIR) {                                                          // unit = (tile-row pair, k tile)
                    const uint32_t tp = u / op.kt, tk = u - tp * op.kt, tn = 2 * tp + crank;
                    valid = tn < tile_rows;                                          // odd N/128: the last pair has one row only
                    tile = tn * op.kt + tk;
                    if (crank == 0) mbar_expect_tx(bar, (2 * tp + 1 < tile_rows) ? 65536 : 32768);
                    bar = map_to_cta(bar, 0);
                } else {
                    mbar_expect_tx(bar, 32768);
                }
                if (!valid) continue;
                const uint64_t off = op.w_offset + (uint64_t)tile * 32768;          // tile index in TILE128 storage order
                const uint32_t slot = __ldg(a.T + (off >> a.log2b));
                const uint64_t byte = ((uint64_t)slot << a.log2b) + (off & ((1ull << a.log2b) - 1));
                const uint32_t row = (uint32_t)(byte >> 8);                          // pool viewed as rows of 256 B
                const uint32_t st = smem_base + s * 32768;
                if (PAIR) {
                    tma_load_2d_pair(st, &map_w, 0, row, bar);
                    tma_load_2d_pair(st + 16384, &map_w, 64, row, bar);
                } else {
                    tma_load_2d(st, &map_w, 0, row, bar);
                    tma_load_2d(st + 16384, &map_w, 64, row, bar);
                }
            }
        }
    } else if (warp == 2 && lane == 0) {
        // ---------------------------------------------------------------- TMA producer, activation tiles (L2-resident)
        gm_dep_wait();
        uint32_t it = 0;
        for (uint32_t j = 0; j < a.nops; ++j) {
            const GemmOp& op = a.ops[j];
            if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;         // this range's part of the op, in op units
            const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
            for (uint32_t u = ubeg; u < uend; ++u, ++it) {
                const uint32_t s = it % a.xstages, f = it / a.xstages;
                if (f > 0) mbar_wait(smem_u32(&xempty[s]), (f - 1) & 1);
                const uint32_t tk = u % op.kt;
                const uint32_t st = x_base + s * xtile;
                uint32_t bar = smem_u32(&xfull[s]);
                if (PAIR) {                                                          // rows [crank * batch/2, +batch/2) of X
                    if (crank == 0) mbar_expect_tx(bar, 2 * xtile);
                    bar = map_to_cta(bar, 0);
                    tma_load_2d_pair(st, &a.map_x[j], tk * 128, crank * (a.batch / 2), bar);
                    tma_load_2d_pair(st + xbox, &a.map_x[j], tk * 128 + 64, crank * (a.batch / 2), bar);
                } else {
                    mbar_expect_tx(bar, xtile);
                    tma_load_2d(st, &a.map_x[j], tk * 128, 0, bar);
                    tma_load_2d(st + xbox, &a.map_x[j], tk * 128 + 64, 0, bar);
                }
            }
        }
    } else if (warp == 1 && lane == 0 && crank == 0) {
        // ---------------------------------------------------------------- MMA issuer (the pair's leader only)
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((a.batch >> 3) << 17) | (((PAIR ? 256u : 128u) >> 4) << 24);
        uint32_t it = 0, seg = 0;                                               // both run on across the ops
        auto acquire_acc = [&]() {                                              // accumulator seg & 1 drained by the epilogue?
            if (seg >= 2) {
                mbar_wait(smem_u32(&tmem_empty[seg & 1]), ((seg >> 1) - 1) & 1);
                tc_fence_after();
            }
        };
        auto commit = [&](uint64_t* bar) {
            if (PAIR) tc_commit_pair(smem_u32(bar));
            else tc_commit(smem_u32(bar));
        };
        for (uint32_t j = 0; j < a.nops; ++j) {
            const GemmOp& op = a.ops[j];
            if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;         // this range's part of the op, in op units
            const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
            uint32_t cur_tn = ubeg / op.kt;
            bool first = true;
            acquire_acc();
            for (uint32_t u = ubeg; u < uend; ++u, ++it) {
                const uint32_t tn = u / op.kt;
                if (tn != cur_tn) {
                    commit(&tmem_full[seg & 1]);                                 // accumulator of the finished tile row (pair)
                    ++seg;
                    cur_tn = tn;
                    first = true;
                    acquire_acc();
                }
                const uint32_t ws = it % a.wstages, xs = it % a.xstages;
                mbar_wait(smem_u32(&xfull[xs]), (it / a.xstages) & 1);
                mbar_wait(smem_u32(&wfull[ws]), (it / a.wstages) & 1);
                tc_fence_after();
                const uint32_t st = smem_base + ws * 32768, sx = x_base + xs * xtile;
                const uint32_t d = tmem_base + (seg & 1) * a.batch;
#pragma unroll
                for (int box = 0; box < 2; ++box) {
                    const uint64_t ad = umma_desc_sw128(st + box * 16384);
                    const uint64_t bd = umma_desc_sw128(sx + box * xbox);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {                                // UMMA_K = 16 bf16 = 32 B inside the atom
                        const uint32_t acc = (first && box == 0 && k == 0) ? 0u : 1u;
                        if (PAIR) tc_mma_bf16_pair(d, ad + 2 * k, bd + 2 * k, idesc, acc);
                        else tc_mma_bf16(d, ad + 2 * k, bd + 2 * k, idesc, acc);
                    }
                }
                first = false;
                commit(&wempty[ws]);                                             // frees both stages when the MMAs retire
                commit(&xempty[xs]);
            }
            commit(&tmem_full[seg & 1]);
            ++seg;
        }
    } else if (warp >= 3) {
        // ---------------------------------------------------------------- epilogue (4 warps = 4 TMEM lane quarters)
        const uint32_t q = warp & 3, r = q * 32 + lane;
        const int etid = threadIdx.x - 96;
        gm_dep_wait();
        if (etid == 0) gm_dep_launch();
        const uint32_t nout = a.batch * 128;
        const uint32_t eb0 = PAIR ? map_to_cta(smem_u32(&tmem_empty[0]), 0) : smem_u32(&tmem_empty[0]);   // the leader's
        const uint32_t eb1 = PAIR ? map_to_cta(smem_u32(&tmem_empty[1]), 0) : smem_u32(&tmem_empty[1]);
        uint32_t seg = 0;
        for (uint32_t j = 0; j < a.nops; ++j) {
            const GemmOp& op = a.ops[j];
            const uint32_t kt = op.kt;
            if (op.ubase + op.units <= gbeg || op.ubase >= gend) continue;         // this range's part of the op, in op units
            const uint32_t ubeg = max(gbeg, op.ubase) - op.ubase, uend = min(gend, op.ubase + op.units) - op.ubase;
            float* part = a.part + op.part_base;
            uint32_t* counters = a.counters + op.row_base;
            for (uint32_t u = ubeg; u < uend; ++seg) {
                const uint32_t tg = u / kt;                                      // tile row, or tile-row pair
                const uint32_t t_first = tg * kt, t_last = t_first + kt - 1;
                const uint32_t seg_last = min(uend - 1, t_last);
                const bool complete = (u == t_first) && (seg_last == t_last);
                const uint32_t tn = PAIR ? 2 * tg + crank : tg;                  // this CTA's tile row
                const bool valid = !PAIR || tn * 128 < op.N;
                mbar_wait(smem_u32(&tmem_full[seg & 1]), (seg >> 1) & 1);
                tc_fence_after();
                const uint32_t taddr = tmem_base + ((q * 32) << 16) + (seg & 1) * a.batch;
                const size_t n = (size_t)tn * 128 + r;
                const uint32_t c_first = (op.ubase + t_first) / a.per, c_last = (op.ubase + t_last) / a.per;   // ranges that meet the row
                const uint32_t ncontrib = c_last - c_first + 1, me = rank_in_grid - c_first;
                float* mine = part + ((size_t)tn * op.maxc + me) * nout;
                const bool finisher = valid && !complete && me == 0;
                if (finisher) {
                    // The row's FIRST contributor finishes it: for that CTA it is the last row of its range, the others met the
                    // row at the start of theirs and have published long before.  (With "last to arrive reduces", whoever
                    // was last fell behind, was last again, and the launch ended with its slowest CTA.)  Its own part never
                    // leaves the chip: TMEM -> registers, + the others' partials in contributor order, -> Y.
                    if (etid == 0) {
                        uint32_t seen;
                        do {
                            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(counters + tn) : "memory");
                            if (seen != ncontrib - 1) __nanosleep(64);
                        } while (seen != ncontrib - 1);
                        counters[tn] = 0;                                        // self-reset for the next launch
                    }
                    epi_bar();
                    __threadfence();
                }
                if (valid) {
                    const float* others = part + ((size_t)tn * op.maxc + 1) * nout + r;      // contributors 1 .. ncontrib-1
                    for (uint32_t c = 0; c < a.batch; c += 16) {
                        uint32_t v[16];
                        if (finisher) {
                            // up to 3 x 16 partial loads in flight per thread beside the TMEM load (L2-latency bound)
                            float sum[16];
                            for (uint32_t p = 0; p + 1 < ncontrib || p == 0; p += 3) {
                                float x[3][16];
#pragma unroll
                                for (int pp = 0; pp < 3; ++pp) {
                                    const float* src = others + (size_t)(p + pp) * nout + (size_t)c * 128;
#pragma unroll
                                    for (int i = 0; i < 16; ++i) x[pp][i] = (p + pp + 1 < ncontrib) ? __ldcg(src + i * 128) : 0.f;
                                }
                                if (p == 0) {
                                    tc_ld16(taddr + c, v);
#pragma unroll
                                    for (int i = 0; i < 16; ++i) sum[i] = __uint_as_float(v[i]);
                                }
#pragma unroll
                                for (int pp = 0; pp < 3; ++pp)
                                    if (p + pp + 1 < ncontrib)
#pragma unroll
                                        for (int i = 0; i < 16; ++i) sum[i] += x[pp][i];
                            }
#pragma unroll
                            for (int i = 0; i < 16; ++i) op.y[(size_t)(c + i) * op.N + n] = __float2bfloat16_rn(sum[i]);
                            continue;
                        }
                        tc_ld16(taddr + c, v);
                        if (complete) {
#pragma unroll
                            for (int i = 0; i < 16; ++i) op.y[(size_t)(c + i) * op.N + n] = __float2bfloat16_rn(__uint_as_float(v[i]));
                        } else {
#pragma unroll
                            for (int i = 0; i < 16; ++i) __stcg(mine + (size_t)(c + i) * 128 + r, __uint_as_float(v[i]));
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (PAIR) mbar_arrive_cluster((seg & 1) ? eb1 : eb0);
                    else mbar_arrive((seg & 1) ? eb1 : eb0);
                }
                if (valid && !complete && me != 0) {                             // publish this CTA's part of the cut row
                    __threadfence();
                    epi_bar();
                    if (etid == 0) asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(counters + tn), "r"(1u) : "memory");
                }
                u = seg_last + 1;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (PAIR) cluster_sync_all();      // the peer's shared memory and barriers stay alive until both CTAs are done
    if (warp == 1) {
        tc_fence_after();
        if (PAIR) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(a.tmem_cols) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(a.tmem_cols) : "memory");
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

extern bool g_gemv_pdl;      // gemv_stream.cu: the PDL A/B switch (cloak_set_gemv_engine(2) turns it off)
cloak_status check_linear(const cloak_pool* pool, const cloak_tensor* w, const void* x, void* y, const char* who);

}  // namespace cloak

using namespace cloak;

namespace cloak {

static cloak_status gemm_check(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y, uint32_t batch,
                               const char* who) {
    cloak_status st = check_linear(pool, w, d_x, d_y, who);
    if (st != CLOAK_OK) return st;
    if (batch < 16 || batch > 256 || batch % 16) return fail(CLOAK_ERR_INVALID, "%s: batch must be a multiple of 16 in 16..256", who);
    if (w->dt != CLOAK_BF16 || w->layout != CLOAK_TILE128) return fail(CLOAK_ERR_UNSUPPORTED, "%s: needs CLOAK_BF16 in CLOAK_TILE128 layout", who);
    if (w->N % 128 || w->K % 128) return fail(CLOAK_ERR_ALIGN, "%s: N and K must be multiples of 128", who);
    if (pool->block < 32768) return fail(CLOAK_ERR_UNSUPPORTED, "%s: block_bytes must be >= 32 KiB (one 128x128 bf16 tile)", who);
    return CLOAK_OK;
}

static int g_gemm_engine = 0;      // 0 auto, 1 one CTA per range, 2 CTA pairs (cloak_set_gemm_engine)

// CTA pairs that can be resident at once (the split-K hand-over spins on other ranges: all of them must be running)
static int max_pairs(int device, int sms) {
    static int cached[64];
    if (device < 0 || device >= 64) return 0;
    if (cached[device]) return cached[device];
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * (sms / 2));
    cfg.blockDim = dim3(GM_THREADS);
    cfg.dynamicSmemBytes = 226 * 1024;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, gemm_tile128_kernel<true>, &cfg) != cudaSuccess) {
        cudaGetLastError();
        n = 0;
    }
    if (n > sms / 2) n = sms / 2;
    cached[device] = n > 0 ? n : -1;
    return cached[device];
}

// One launch of n <= GM_MAX_OPS checked ops.
static cloak_status gemm_launch(const cloak_pool* pool, const cloak_gemm_op* ops, uint32_t n, uint32_t batch, cudaStream_t s) {
    cloak_status st;
    if (!pool->tmap_ready) {
        cloak_pool* p = const_cast<cloak_pool*>(pool);
        st = make_map(&p->tmap_tile128, pool->base, 128, pool->bytes() / 256, 256, 64, 128);
        if (st != CLOAK_OK) return st;
        p->tmap_ready = true;
    }
    static bool attr_set = false;
    if (!attr_set) {
        CLOAK_CUDA(cudaFuncSetAttribute(gemm_tile128_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024));
        CLOAK_CUDA(cudaFuncSetAttribute(gemm_tile128_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024));
        attr_set = true;
    }
    GemmArgs a;
    a.T = pool->d_T;
    a.log2b = pool->log2_block;
    a.batch = batch;
    a.nops = n;
    const int sms = sm_count(pool->device);
    // CTA pairs from batch 64 on: the X tile is then at least half a W tile, and sharing it between two tile rows pays
    bool pair = g_gemm_engine == 2 || (g_gemm_engine == 0 && batch >= 64);
    int ranges = sms;                   // ranges per op: one per CTA or per pair
    if (pair) {
        ranges = max_pairs(pool->device, sms);
        if (ranges <= 0) {
            pair = false;
            ranges = sms;
        }
    }
    uint32_t cap = 512 / batch;         // contributors per tile row (fp32 partials are batch * 512 B each): ~10 at batch 32, 4 at 128
    cap = cap < 4 ? 4 : (cap > 10 ? 10 : cap);
    // The launch's units -- all ops back to back, each tn-major -- are cut into equal contiguous ranges, one per CTA (pair):
    // a range boundary costs one tile row of fp32 partials and one reduction, and there are ranges - 1 of them per
    // LAUNCH, wherever the op boundaries fall (cut per op it was ranges - 1 per op: 14 x the partial traffic and the
    // reductions for the 14 projections of two layers, and ops with few units left CTAs idle).
    uint64_t rows = 0, total = 0;
    uint32_t max_kt = 0;
    for (uint32_t j = 0; j < n; ++j) {
        const cloak_tensor& w = ops[j].w;
        st = make_map(&a.map_x[j], ops[j].d_x, w.K, batch, (uint64_t)w.K * 2, 64, pair ? batch / 2 : batch);
        if (st != CLOAK_OK) return st;
        GemmOp& o = a.ops[j];
        o.w_offset = w.w_offset;
        o.y = static_cast<__nv_bfloat16*>(ops[j].d_y);
        o.N = w.N;
        o.kt = w.K / 128;
        const uint32_t tile_rows = w.N / 128;
        const uint64_t units64 = (uint64_t)(pair ? (tile_rows + 1) / 2 : tile_rows) * o.kt;   // pair: (tile-row pair, k tile)
        if (total + units64 > 0xffffffffull) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: too many tiles in one launch");
        o.units = (uint32_t)units64;
        o.ubase = (uint32_t)total;
        o.row_base = (uint32_t)rows;
        total += units64;
        rows += tile_rows;
        if (o.kt > max_kt) max_kt = o.kt;
    }
    uint32_t per = (uint32_t)((total + ranges - 1) / ranges);
    if (per < (max_kt + cap - 1) / cap) per = (max_kt + cap - 1) / cap;     // at most ~cap ranges meet one tile row
    const uint32_t ctas = (uint32_t)((total + per - 1) / per);
    a.per = per;
    a.total = (uint32_t)total;
    uint64_t part = 0;
    for (uint32_t j = 0; j < n; ++j) {
        GemmOp& o = a.ops[j];
        o.maxc = (o.kt + per - 1) / per + 1;
        o.part_base = part;
        part += (uint64_t)(o.N / 128) * o.maxc * batch * 128;
    }
    if (rows * 4 > WS_COUNTER_BYTES) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: too many output rows for the tile counters");
    const uint32_t xtile = (pair ? batch / 2 : batch) * 256;     // per CTA
    a.xstages = 2;
    uint32_t wst = (224u * 1024u - a.xstages * xtile) / 32768u;
    if (wst > GM_MAX_STAGES) wst = GM_MAX_STAGES;
    if (wst < 2) return fail(CLOAK_ERR_UNSUPPORTED, "gemm: batch too large for the shared-memory ring");
    a.wstages = wst;
    a.tmem_cols = 32;
    while (a.tmem_cols < 2 * batch) a.tmem_cols <<= 1;
    st = pool_workspace(pool, WS_COUNTER_BYTES + part * 4);
    if (st != CLOAK_OK) return st;
    a.counters = reinterpret_cast<uint32_t*>(pool->ws);
    a.part = reinterpret_cast<float*>(pool->ws + WS_COUNTER_BYTES);

    const size_t smem = (size_t)a.wstages * 32768 + (size_t)a.xstages * xtile + 1024;
    a.early = (g_gemv_pdl && !pool->dirty) ? 1u : 0u;
    if (pool->dirty && pool->dirty_stream == s) pool->dirty = false;   // this launch waits for the writer in full
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(pair ? 2 * ctas : ctas);
    cfg.blockDim = dim3(GM_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[2];
    unsigned na = 0;
    if (pair) {
        at[na].id = cudaLaunchAttributeClusterDimension;
        at[na].val.clusterDim.x = 2;
        at[na].val.clusterDim.y = 1;
        at[na].val.clusterDim.z = 1;
        ++na;
    }
    if (g_gemv_pdl) {
        at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    if (pair) CLOAK_CUDA(cudaLaunchKernelEx(&cfg, gemm_tile128_kernel<true>, pool->tmap_tile128, a));
    else CLOAK_CUDA(cudaLaunchKernelEx(&cfg, gemm_tile128_kernel<false>, pool->tmap_tile128, a));
    launched();
    return CLOAK_OK;
}

}  // namespace cloak

extern "C" cloak_status cloak_set_gemm_engine(int engine) {
    if (engine < 0 || engine > 2) return fail(CLOAK_ERR_INVALID, "set_gemm_engine: engine must be 0, 1 or 2");
    g_gemm_engine = engine;
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

extern "C" cloak_status cloak_gemm_chain(const cloak_pool* pool, const cloak_gemm_op* h_ops, uint32_t n_ops, uint32_t batch,
                                         void* stream) {
    if (!h_ops || n_ops == 0) return fail(CLOAK_ERR_INVALID, "gemm_chain: no ops");
    for (uint32_t i = 0; i < n_ops; ++i) {
        cloak_status st = gemm_check(pool, &h_ops[i].w, h_ops[i].d_x, h_ops[i].d_y, batch, "gemm_chain");
        if (st != CLOAK_OK) return st;
    }
    DeviceGuard g(pool->device);
    for (uint32_t i = 0; i < n_ops;) {                      // at most GM_MAX_OPS ops and 2^18 tile rows per launch
        uint32_t n = 0;
        uint64_t rows = 0;
        while (i + n < n_ops && n < (uint32_t)GM_MAX_OPS && rows + h_ops[i + n].w.N / 128 <= 200000) rows += h_ops[i + n++].w.N / 128;
        if (n == 0) return fail(CLOAK_ERR_UNSUPPORTED, "gemm_chain: op %u has too many output rows", i);
        cloak_status st = gemm_launch(pool, h_ops + i, n, batch, (cudaStream_t)stream);
        if (st != CLOAK_OK) return st;
        i += n;
    }
    return CLOAK_OK;
}
