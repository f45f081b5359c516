// S6 cloak_gemv / cloak_gemv_chain, bf16, K % 256 == 0: the streaming (persistent, TMA-fed) kernel.
//
// Same contraction and table translation as gemv.cu (north_star (c)), organised for the
// HBM roofline.  Measured on B200: a pure stream of 16 x 2 KiB row pieces per stage tops out
// at 5.5 TB/s, 8 x 4 KiB pieces at 6.4 TB/s, so a unit of work is (8 weight rows) x (CB of each row), CB = the largest
// multiple of 512 B up to 4 KiB that divides the row (4 KiB for every LLaMA / Qwen projection but a few):
//   * one persistent CTA per SM; an op's units are numbered tile-major (u = tile * kch + chunk) and cut into
//     contiguous ranges equal to within one unit, one per CTA (stream-K); the ranges that are one unit longer go, op after op,
//     to the CTAs that hold the least so far: every SM moves the same bytes to within a unit or two, no wave tail;
//   * warp 0 produces: 8 lanes each translate one row piece through the block table and issue one
//     cp.async.bulk (TMA 1-D) into a shared-memory ring (6 stages of 32 KiB), completion on an mbarrier;
//   * eight consumer warps (behind the producer and the helper warp): each owns one eighth of the k-range of a chunk.  The weights are the B operand of
//     mma.sync.m16n8k16 (8 weight rows = N), the activations the A operand (batch rows = M, zero-padded to 8 or
//     16).  Lane (g, t) reads one 16-byte vector of weight row g per 64-byte step; since a contraction may visit
//     k in any order, the vector's elements are *declared* to be the MMA's k-slots (2t, 2t+1, 2t+8, 2t+9) and
//     X is loaded by the same rule: both operands are plain 16-byte loads, no transposes;
//   * inside its range a CTA walks groups of TG = 8 row tiles chunk-major (all tiles of the group for chunk 0,
//     then chunk 1, ...), so a warp's X fragments are fetched once per (group, chunk) and reused for 64 weight
//     rows: X traffic from L2 is batch/64 of the weight traffic;
//   * accumulators (one m16n8 tile per row tile of the group, two interleaved to halve the dependency chain)
//     stay in registers until the group is done, are reduced over the 8 warps in shared memory, and stored.
//   * a row tile cut by a range boundary is finished by its OWNER, the CTA that holds the tile's first unit (for
//     which it is the last tile of the range).  Every other contributor meets the tile first, publishes its fp32
//     partial early (release), and moves on; the owner, done with everything else, waits for those arrivals
//     (acquire; all CTAs are co-resident, one per SM) and adds the partials in contributor order:
//     deterministic, and bit-identical between a cloaked and an identity-table pool, which differ only in
//     addresses.  No fence, atomic round trip or reduction sits at the end of the other CTAs.
//   * all of that device-scope work -- the release that publishes a partial, the owner's acquire-wait, its partial loads and
//     stores, the report that an op is done -- is done by a HELPER warp (warp 1), to which the consumers post records through a
//     small shared-memory queue: while consumer warps sit in an L2 round trip no ring stage is handed back and no copy is issued
//     (measured: 7.8 of 80.9 us for the 7 ops of the cfg1 layer; see GS_NREC).
//   * a launch executes a CHAIN of ops (cloak_gemv_chain; cloak_gemv is a chain of one).  The producer warp
//     runs straight through the chain -- weights do not depend on activations -- so HBM stays busy across op
//     boundaries (an op with fewer ranges than CTAs starts at the CTA where the previous one stopped when such ops
//     dominate the launch); only the consumers of an op marked `after` wait, on a grid-wide arrival counter, for all CTAs
//     to have finished the earlier ops (its X is their Y); several ops can share one such arrival.  An op may also emit silu(G) * Y next to Y in its
//     epilogue (the gated MLP's activation, O9), where G is the output of an earlier op of the same shape -- the
//     same CTA wrote those very elements, so no wait is needed -- and gate/up -> down costs no separate pass.
//   * programmatic dependent launch: the grid may start while its stream predecessor drains; the producer
//     streams W (immutable during decode) ahead of griddepcontrol.wait, everything else waits.
//   * fusion of small ops (batch <= 8; plan_fusion, the SEG = true instantiations): independent ops of one shape whose rows are a
//     single chunk -- the selected experts' projections of an MoE layer, 96 units for 148 CTAs each -- are dealt out as ONE op over
//     the concatenation of their row tiles (a segment table in the kernel parameters), each tile fetched with one bulk copy
//     (its 8 rows are contiguous in the arena).  Same sums in the same order: bit-identical to the unfused launch.
//   * cloak_gemv_static (end of this file): the same kernel with its scratch in a fixed static device array -- allocates nothing.
#include <cuda_bf16.h>
#include <type_traits>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

struct ChainOp {             // 88 bytes of kernel parameter space per op (11 x 8)
    uint64_t w_offset;
    const uint16_t* x;       // [batch, K]
    __nv_bfloat16* y;        // [batch, N]
    const uint16_t* gate;    // NULL, or [batch, N] written by an earlier op with the same (N, K): then also
    uint16_t* act;           //   act[m, n] = silu(gate[m, n]) * y[m, n]   (O9, the gated MLP's activation)
    uint32_t N, K;
    uint32_t kch;            // chunks per row = K*2 / CB
    uint32_t units;          // tiles * kch
    uint32_t per;            // units per range: range r (of min(units, grid) ranges) starts at r * per + min(r, rem) and holds
    uint32_t rem;            //   per + (r < rem) units -- equal to within one unit
    uint32_t ctas;           // ranges = CTAs that own units of this op (host side only)
    uint32_t pad_;
    uint32_t tile_base;      // index of this op's first row-tile counter
    uint32_t flags;          // OP_SIGNAL
    uint32_t wait_op;        // NO_WAIT, or the index of the op whose completion by ALL CTAs this op's consumers wait for
    uint32_t rot;            // range r of this op belongs to CTA (r + rot) % grid: an op with fewer ranges than CTAs starts
                             // where the previous one stopped, so the idle CTAs are different ones each time (an op with a
                             // gate epilogue keeps the rotation of the op that produced the gate: same rows, same CTA)
};
enum { OP_SIGNAL = 2 };      // some later op waits for this one: every CTA reports here when it is done with it (and all before)
constexpr uint32_t NO_WAIT = 0xffffffffu;
constexpr int GS_MAX_OPS = 48;              // 48 x 80 B + header < 4 KiB of kernel parameters

struct ChainArgs {
    const char* pool;
    const uint32_t* T;
    float* part;             // [op][cta][batch * 8]: partial of the cut row tile a CTA meets first in that op
    uint32_t* counters;      // [tile_base + tile]: arrivals of the non-owning contributors; owner resets to 0
    uint32_t* opsync;        // [GS_MAX_OPS] arrivals per signalling op, [GS_MAX_OPS] CTAs done with the launch: the last resets all
    unsigned long long* trace;   // NULL, or [gridDim.x][4]: %smid, globaltimer at CTA start, producer done, consumers done
    uint32_t log2b;
    uint32_t batch;
    uint32_t nops;
    uint32_t early;          // 1: W is unchanged since before the preceding kernel, so the producer may stream it
                             //    ahead of griddepcontrol.wait (programmatic dependent launch)
    uint32_t any_signal;     // some op of this launch signals
    ChainOp ops[GS_MAX_OPS];
};

// Segmented ops (SEG kernels, batch <= 8): an op whose row tiles come from several matrices of one shape -- the selected experts'
// gate (or up, or down) projections of an MoE layer, fused by the host into ONE op of nseg x (N / 8) tiles so that a CTA streams
// several units per op instead of at most one (gemv_stream_launch: fusion).  Tile t of the op is tile t % tps of segment t / tps.
struct ChainSeg {
    uint64_t w_offset;
    const uint16_t* x;
    __nv_bfloat16* y;
    const uint16_t* gate;
    uint16_t* act;
};
struct ChainArgsSeg {
    ChainArgs base;                  // ops[j].N / K are one segment's; units = nseg * tps * kch; w_offset, x, y, gate, act unused
    ChainSeg segs[GS_MAX_OPS];       // every original op of the launch is a segment of exactly one fused op
    uint32_t tps[GS_MAX_OPS];        // tiles per segment of op j (N / 8)
    uint32_t seg0[GS_MAX_OPS];       // op j's first entry in segs[]
};
__device__ __forceinline__ const ChainArgs& chain_base(const ChainArgs& a) { return a; }
__device__ __forceinline__ const ChainArgs& chain_base(const ChainArgsSeg& a) { return a.base; }

constexpr int GS_CONSUMERS = 8;                       // consumer warps
// Warps ahead of the consumers.  batch <= 8: the producer warp and the helper warp.  batch 9..16: a whole warpgroup (producer,
// helper and two warps that retire at once), so that the register file can be re-split per warpgroup with setmaxnreg: the lead
// group drops to 56 registers per thread, the two consumer groups rise to 224 -- room for a second set of X fragments.
constexpr int gs_lead_warps(int nt) { return nt == 2 ? 4 : 2; }      // warp 0 = producer, warp 1 = helper (see GS_NREC)
constexpr int gs_threads(int nt) { return 32 * (gs_lead_warps(nt) + GS_CONSUMERS); }
constexpr int GS_ROWS = 8;                            // weight rows per tile (the MMA's N)
constexpr int GS_PAD = 64;                            // bytes of padding per staged row (conflict-free LDS.128)
// Row tiles per group (X reuse; one register accumulator set per tile) and interleaved accumulators per tile.
// 8 tiles x 2 accumulators measured best for both batch ranges: 16 x 1 halves the X traffic at batch 16 but its
// 16-deep dependent MMA chain costs more than that saves; staggering the group boundaries over the CTAs (so the
// SMs do not all wait for X at once) adds a group per CTA and was slower too.
// (With the X prefetch in place at batch 9..16, 16 x 1, 12 x 1 and 12 x 2 were measured again: 94.5, 96.1, 101.4 us for the
// cfg1 layer against 93.6 us for 8 x 2.)
constexpr int gs_tg(int) { return 8; }
constexpr int gs_nacc(int) { return 2; }
constexpr int GS_TGR = 4;                             // row tiles reduced across warps per shared-memory pass
constexpr int GS_MAX_STAGES = 12;
// The HELPER warp.  Everything a CTA does at device scope for other CTAs -- publishing the partial of a cut head tile (a release),
// finishing the cut tail tile it owns (an acquire-wait for the other contributors, their partials, the stores), reporting an op
// done (a release) -- costs an L2 round trip or more, and while the consumer warps sit in it no ring stage is handed back, so no
// new copy is issued: measured on the cfg1 layer, 7 ops, batch 1, those two epilogues cost 7.8 of 80.9 us (one op of the same
// bytes: 70.0 us).  The consumers therefore only POST such work -- a record in a small shared-memory queue (mbarrier full / empty
// per slot; the tail tile's own sums travel in the slot) -- and go on streaming; warp 1 executes the records in order.
constexpr int GS_NREC = 8;
enum { REC_PUBLISH = 0, REC_TAIL = 1, REC_SIGNAL = 2, REC_EXIT = 3 };
struct HelperRec { uint32_t kind, j, tile, nc, vr; };
constexpr uint32_t gs_stages(int cu) {                // cu = chunk bytes / 512; ~192 KiB of weights in flight per SM
    return 196608u / (GS_ROWS * cu * 512u) > GS_MAX_STAGES ? GS_MAX_STAGES : 196608u / (GS_ROWS * cu * 512u);
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
// Activations may have been written earlier in this same kernel by other SMs (an OP_AFTER op reads its
// predecessors' Y): a coherent load, ordered behind the acquire that ended the grid-wide wait -- never ld.global.nc.
__device__ __forceinline__ uint4 ldg_coherent(const void* p) {
    uint4 r;
    asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(uint32_t* p, uint32_t v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
// Programmatic dependent launch (PDL): this grid may start while its stream predecessor is still draining.
// grid_dep_wait returns once the predecessor has completed and its writes are visible; grid_dep_launch lets the
// stream successor start.  Every kernel here triggers only AFTER its own wait, so whatever a successor does ahead
// of its wait still observes everything older than its immediate predecessor.
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ uint32_t my_smid() {
    uint32_t s;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(s));
    return s;
}
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" :: "n"(GS_CONSUMERS * 32) : "memory"); }

// silu(g) * u for bf16 inputs, fp32 arithmetic, round to nearest even: bit for bit cloak_silu_mul's result.
__device__ __forceinline__ uint16_t silu_mul_bf16(uint16_t g, __nv_bfloat16 u) {
    const float z = __uint_as_float((uint32_t)g << 16), w = __bfloat162float(u);
    uint32_t b = __float_as_uint(z / (1.0f + __expf(-z)) * w);
    b += 0x7FFFu + ((b >> 16) & 1u);
    return (uint16_t)(b >> 16);
}
__device__ __forceinline__ uint16_t ld_coherent_u16(const uint16_t* p) {
    uint16_t v;
    asm volatile("ld.global.u16 %0, [%1];" : "=h"(v) : "l"(p) : "memory");
    return v;
}

// CU: chunk bytes per row / 512 (1..8; the largest divisor of the row's 512-byte units that is <= 8, so a 10 KiB row is cut
// into 2.5 KiB chunks and a 1.5 KiB row is one chunk -- larger TMA pieces than a power of two would allow).
// NT: 1 = batch <= 8 (upper half of the MMA's M is zero), 2 = batch <= 16.
template <int CU, int NT, bool SEG = false>
__global__ void __launch_bounds__(gs_threads(NT), 1)
gemv_chain_kernel(const __grid_constant__ typename std::conditional<SEG, ChainArgsSeg, ChainArgs>::type args) {
    const ChainArgs& a = chain_base(args);
    constexpr uint32_t CB = CU * 512u;
    constexpr uint32_t RS = CB + GS_PAD;                       // staged row stride
    constexpr uint32_t STAGE = GS_ROWS * RS;
    constexpr uint32_t NST = gs_stages(CU);
    constexpr int KS = CB / (GS_CONSUMERS * 64);               // 64-byte steps (one 16-byte vector per lane) per warp per unit
    constexpr bool PF = (NT == 2);                             // prefetch the next phase's X fragments (see below)
    constexpr int LEAD = gs_lead_warps(NT);
    constexpr int GS_TG = gs_tg(NT), GS_NACC = gs_nacc(NT);
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full[NST], empty[NST];
    __shared__ float red[GS_CONSUMERS][GS_TGR][NT * 64];      // [warp][tile][batch m][row r]
    __shared__ float own[GS_NREC][NT * 64];                    // per helper record: this CTA's own sums of the cut tile it owns
    __shared__ HelperRec rec[GS_NREC];
    __shared__ __align__(8) uint64_t rec_full[GS_NREC], rec_empty[GS_NREC];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
#pragma unroll
        for (uint32_t s = 0; s < NST; ++s) {
            mbar_init(smem_u32(&full[s]), 1);
            mbar_init(smem_u32(&empty[s]), GS_CONSUMERS);
        }
#pragma unroll
        for (int r = 0; r < GS_NREC; ++r) {
            mbar_init(smem_u32(&rec_full[r]), 1);
            mbar_init(smem_u32(&rec_empty[r]), 1);
        }
        fence_barrier_init();
    }
    __syncthreads();
    const uint32_t smem_base = smem_u32(smem);

    // Every Y element is stored exactly once, by the CTA that owns its row tile (its consumers, or its helper for a cut tail tile).
    // The gate op had the same (N, K), hence the same split: gate[idx] was stored by this CTA -- by the same role -- before.
    // store_out(j, tile, m, r, sum): batch row m, row r of row tile `tile` of op j.
    auto store_out = [&](uint32_t j, uint32_t tile, uint32_t m, uint32_t r, float sum) {
        const ChainOp& op = a.ops[j];
        const __nv_bfloat16 v = __float2bfloat16_rn(sum);
        if constexpr (SEG) {
            const uint32_t sg = tile / args.tps[j];
            const ChainSeg& sgm = args.segs[args.seg0[j] + sg];
            const size_t idx = (size_t)m * op.N + (tile - sg * args.tps[j]) * GS_ROWS + r;
            sgm.y[idx] = v;
            if (sgm.gate) sgm.act[idx] = silu_mul_bf16(ld_coherent_u16(sgm.gate + idx), v);
        } else {
            const size_t idx = (size_t)m * op.N + tile * GS_ROWS + r;
            op.y[idx] = v;
            if (op.gate) op.act[idx] = silu_mul_bf16(ld_coherent_u16(op.gate + idx), v);
        }
    };

    if (warp < LEAD) {
        if (NT == 2) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 1) {
            // -------------------------------------------------------- helper: the CTA's device-scope work, in the order posted
            grid_dep_wait();                                 // counters, partials and Y belong to stream order
            const uint32_t nout = a.batch * GS_ROWS;
            for (uint32_t hs = 0;; ++hs) {
                const uint32_t slot = hs % GS_NREC;
                mbar_wait(smem_u32(&rec_full[slot]), (hs / GS_NREC) & 1);
                const HelperRec r = rec[slot];
                if (r.kind == REC_PUBLISH) {
                    // the consumers' partial stores are ordered before this by their barrier and the slot's mbarrier: the release is cumulative
                    if (lane == 0) red_release_add(a.counters + a.ops[r.j].tile_base + r.tile, 1u);
                } else if (r.kind == REC_TAIL) {
                    // owner of the tail tile: wait for the other contributors (the CTAs after this one), add in CTA order
                    uint32_t* cnt = a.counters + a.ops[r.j].tile_base + r.tile;
                    if (lane == 0) {
                        while (ld_acquire(cnt) != r.nc) __nanosleep(32);
                        *cnt = 0;                                   // self-reset for the next launch
                    }
                    __syncwarp();
                    const float* mypart = a.part + ((size_t)r.j * gridDim.x + r.vr) * nout;
                    for (uint32_t i = lane; i < nout; i += 32) {
                        float sum = own[slot][i];
                        for (uint32_t q = 1; q <= r.nc; ++q) sum += __ldcg(mypart + (size_t)q * nout + i);
                        store_out(r.j, r.tile, i / GS_ROWS, i % GS_ROWS, sum);
                    }
                } else if (r.kind == REC_SIGNAL) {
                    // this CTA is done with op j and everything before it (Y stores: the consumers' before their barrier, the tails' above)
                    __syncwarp();
                    if (lane == 0) red_release_add(a.opsync + r.j, 1u);
                } else {
                    // the arrival counters are reset for the next launch by the last CTA to get here (nobody reads them any more)
                    if (a.any_signal && lane == 0) {
                        if (atomicAdd(a.opsync + GS_MAX_OPS, 1u) == gridDim.x - 1) {
                            for (uint32_t j = 0; j < a.nops; ++j) a.opsync[j] = 0;
                            a.opsync[GS_MAX_OPS] = 0;
                        }
                    }
                    return;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&rec_empty[slot]));
            }
        }
        if (warp > 0) return;
        // ------------------------------------------------------------ producer: straight through the chain
        // The table is immutable after cloak_pool_create; the weights may have been written by the preceding
        // kernel (a shuffle / re-layout) unless the host says otherwise.
        if (!a.early) grid_dep_wait();
        uint32_t s = 0, ph = 0;
        bool wrapped = false;
        for (uint32_t j = 0; j < a.nops; ++j) {
            const ChainOp& op = a.ops[j];
            const uint32_t kch = op.kch;
            const uint32_t vr = (blockIdx.x + gridDim.x - op.rot) % gridDim.x;   // this CTA's range of the op
            const uint32_t ubeg = vr * op.per + min(vr, op.rem), uend = min(ubeg + op.per + (vr < op.rem ? 1u : 0u), op.units);
            if (ubeg >= uend) continue;
            const uint32_t tile_lo = ubeg / kch, tile_hi = (uend - 1) / kch;
            const uint64_t row_bytes = (uint64_t)op.K * 2;
            for (uint32_t g0 = tile_lo; g0 <= tile_hi; g0 += GS_TG) {
                const uint32_t g1 = min(g0 + GS_TG - 1, tile_hi);
                for (uint32_t c = 0; c < kch; ++c) {
                    for (uint32_t tile = g0; tile <= g1; ++tile) {
                        const uint32_t u = tile * kch + c;
                        if (u < ubeg || u >= uend) continue;
                        if (wrapped) mbar_wait(smem_u32(&empty[s]), ph ^ 1);
                        const uint32_t bar = smem_u32(&full[s]);
                        if (lane == 0) mbar_expect_tx(bar, GS_ROWS * CB);
                        __syncwarp();
                        // SEG kernels, rows of one chunk: the 8 rows of a tile are CONTIGUOUS in the arena, so the tile comes as one
                        // bulk copy per block touched (unpadded in the stage: 2-way conflicts on the consumers' LDS.128, which have the
                        // slack) instead of 8 row pieces -- the TMA's throughput falls with the piece size (2 KiB pieces: 4.1 TB/s,
                        // 4 KiB: 6.4 TB/s).  The experts' down projections (1.5 KiB rows): 0.38 -> 0.53 of the peak.
                        const bool whole_tile = SEG && kch == 1;
                        if (lane < (whole_tile ? 1 : GS_ROWS)) {
                            // a chunk that is not a power of two may cross a block boundary: one bulk copy per block touched
                            uint64_t woff = op.w_offset;
                            uint32_t lt = tile;                                        // the tile inside its matrix
                            if constexpr (SEG) {
                                const uint32_t sg = tile / args.tps[j];
                                lt = tile - sg * args.tps[j];
                                woff = args.segs[args.seg0[j] + sg].w_offset;
                            }
                            uint64_t off = woff + (uint64_t)(lt * GS_ROWS + lane) * row_bytes + (uint64_t)c * CB;
                            uint32_t dst = smem_base + s * STAGE + lane * RS, left = whole_tile ? GS_ROWS * CB : CB;
                            if (!whole_tile && (CU & (CU - 1)) == 0 && CB <= (1u << a.log2b)) {       // power of two within a block: one copy
                                const uint32_t slot = __ldg(a.T + (off >> a.log2b));
                                bulk_g2s(dst, a.pool + ((uint64_t)slot << a.log2b) + (off & ((1ull << a.log2b) - 1)), CB, bar);
                                left = 0;
                            }
                            while (left) {
                                const uint64_t in_block = off & ((1ull << a.log2b) - 1);
                                const uint64_t room = (1ull << a.log2b) - in_block;
                                const uint32_t n = room < left ? (uint32_t)room : left;
                                const uint32_t slot = __ldg(a.T + (off >> a.log2b));
                                bulk_g2s(dst, a.pool + ((uint64_t)slot << a.log2b) + in_block, n, bar);
                                off += n;
                                dst += n;
                                left -= n;
                            }
                        }
                        if (++s == NST) { s = 0; ph ^= 1; wrapped = true; }
                    }
                }
            }
        }
        if (a.trace && lane == 0) a.trace[4 * blockIdx.x + 2] = global_ns();
        return;
    }

    // ---------------------------------------------------------------- consumers
    if (NT == 2) asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    const int cw = warp - LEAD;
    const int g = lane >> 2, t = lane & 3;
    const uint32_t ctid = threadIdx.x - 32 * LEAD;                 // 0..255 among consumers
    const bool xv0 = (uint32_t)g < a.batch, xv1 = (uint32_t)(g + 8) < a.batch;
    const uint32_t lane_off = cw * (CB / GS_CONSUMERS) + t * 16;   // byte offset of this lane inside a row chunk
    const uint32_t nout = a.batch * GS_ROWS;

    // X, Y, partials and counters all belong to stream order: nothing below touches them before the predecessor
    // has completed.  Meanwhile the producer is already filling the ring.
    const unsigned long long t_start = a.trace ? global_ns() : 0ull;
    grid_dep_wait();
    if (ctid == 0) grid_dep_launch();

    // records for the helper warp: every consumer thread counts them (the conditions are uniform), thread 0 waits for a slot
    // to be free and fills it.  reserve() must be followed by a consumer barrier before anybody else touches own[slot].
    uint32_t rs = 0;
    auto reserve = [&]() {
        const uint32_t slot = rs % GS_NREC;
        if (ctid == 0 && rs >= (uint32_t)GS_NREC) mbar_wait(smem_u32(&rec_empty[slot]), ((rs / GS_NREC) - 1) & 1);
        ++rs;
        return slot;
    };
    auto post = [&](uint32_t slot, uint32_t kind, uint32_t j, uint32_t tile, uint32_t nc, uint32_t vr) {
        if (ctid == 0) {                     // (behind a consumer barrier: everything the record refers to has been written)
            rec[slot].kind = kind;
            rec[slot].j = j;
            rec[slot].tile = tile;
            rec[slot].nc = nc;
            rec[slot].vr = vr;
            mbar_arrive(smem_u32(&rec_full[slot]));
        }
    };

    // X fragments of this warp's k-slice, two register sets (see "X fragments of one phase" below); they outlive an op
    uint4 xa[KS], xb[KS], na[KS], nb[KS];
    const uint16_t* held_x = nullptr;            // batch 9..16: the X whose chunks 0 and 1 sit in (xa, xb) and (na, nb)

    uint32_t s = 0, ph = 0;
    for (uint32_t j = 0; j < a.nops; ++j) {
        const ChainOp& op = a.ops[j];
        const uint32_t kch = op.kch, per = op.per;
        const uint32_t vr = (blockIdx.x + gridDim.x - op.rot) % gridDim.x;       // this CTA's range of the op
        const uint32_t ubeg = vr * per + min(vr, op.rem), uend = min(ubeg + per + (vr < op.rem ? 1u : 0u), op.units);
        const bool have = ubeg < uend;

        if (have && op.wait_op != NO_WAIT) {
            // grid-wide wait: every CTA has reported at op wait_op, i.e. has finished that op and all ops before it
            if (ctid == 0)
                while (ld_acquire(a.opsync + op.wait_op) != gridDim.x) __nanosleep(32);
            consumer_bar();
            held_x = nullptr;                    // X may have been written inside this launch: nothing held is good any more
        }

        if (have) {
            const uint32_t tile_lo = ubeg / kch, tile_hi = (uend - 1) / kch;
            // A cut tile at the head of the range is owned by an earlier CTA (publish our partial); one at the tail
            // is ours to finish, unless the range lies inside a single tile that started before us.
            const bool cut_head = ubeg > tile_lo * kch;
            const bool cut_tail = uend < (tile_hi + 1) * kch && !(tile_hi == tile_lo && cut_head);
            const uint16_t* x0 = op.x + (size_t)g * op.K + lane_off / 2;            // (SEG: set per group, from its segment)
            const uint16_t* x1 = op.x + (size_t)(g + 8) * op.K + lane_off / 2;
            float* mypart = a.part + ((size_t)j * gridDim.x + vr) * nout;
            // X fragments of one (group, chunk) phase.  Batch <= 8 re-reads them mostly from L1; batch 9..16 (X is up to
            // 16 x K x 2 B, more than the L1 left beside the ring) pays an L2 round trip per phase, so there the next
            // phase's fragments are fetched one phase ahead (PF) into a second register set (see gs_lead_warps).
            // Batch 9..16, rows of TWO chunks (K = 4096 at 4 KiB chunks): both chunks' fragments fit the two register sets, so they
            // are loaded once per X -- consecutive ops that read the same activations (q, k, v; gate, up) and all their groups
            // share them -- instead of once per phase: the SMs' ingest is what bounds batch 16.
            const bool resident = PF && kch == 2;
            auto load_x = [&](uint4 (&pa)[KS], uint4 (&pb)[KS], uint32_t c) {
                const uint32_t xk = c * (CB / 2);
                const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
                for (int ks = 0; ks < KS; ++ks) {
                    pa[ks] = xv0 ? ldg_coherent(x0 + xk + ks * 32) : z;
                    pb[ks] = (NT == 2 && xv1) ? ldg_coherent(x1 + xk + ks * 32) : z;
                }
            };
            if (resident) {
                if (held_x != x0) {
                    load_x(xa, xb, 0);
                    load_x(na, nb, 1);
                    held_x = x0;
                }
            } else if (PF) {
                load_x(xa, xb, 0);
                held_x = nullptr;
            }

            for (uint32_t g0 = tile_lo, gnext; g0 <= tile_hi; g0 = gnext) {
                uint32_t g1 = min(g0 + GS_TG - 1, tile_hi);
                if constexpr (SEG) {                               // a group shares X fragments: it stays inside one segment
                    const uint32_t sg = g0 / args.tps[j];
                    g1 = min(g1, (sg + 1) * args.tps[j] - 1);
                    const uint16_t* xs = args.segs[args.seg0[j] + sg].x;
                    x0 = xs + (size_t)g * op.K + lane_off / 2;
                    x1 = xs + (size_t)(g + 8) * op.K + lane_off / 2;
                }
                gnext = SEG ? g1 + 1 : g0 + GS_TG;
                float acc[GS_TG][GS_NACC][4];
#pragma unroll
                for (int q = 0; q < GS_TG; ++q)
#pragma unroll
                    for (int n = 0; n < GS_NACC; ++n)
#pragma unroll
                        for (int i = 0; i < 4; ++i) acc[q][n][i] = 0.f;

                // one (group, chunk) phase: the group's row tiles of chunk c against the fragments (pa, pb)
                auto phase = [&](const uint4 (&pa)[KS], const uint4 (&pb)[KS], uint32_t c) {
#pragma unroll
                    for (int q = 0; q < GS_TG; ++q) {
                        const uint32_t tile = g0 + q, u = tile * kch + c;
                        if (tile > g1 || u < ubeg || u >= uend) continue;
                        mbar_wait(smem_u32(&full[s]), ph);
                        const uint32_t base = smem_base + s * STAGE + g * ((SEG && kch == 1) ? CB : RS) + lane_off;
#pragma unroll
                        for (int ks = 0; ks < KS; ++ks) {
                            const uint4 w = lds128(base + ks * 64);
                            mma_16816(acc[q][0], pa[ks].x, pb[ks].x, pa[ks].y, pb[ks].y, w.x, w.y);
                            mma_16816(acc[q][GS_NACC - 1], pa[ks].z, pb[ks].z, pa[ks].w, pb[ks].w, w.z, w.w);
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(smem_u32(&empty[s]));
                        if (++s == NST) { s = 0; ph ^= 1; }
                    }
                };
                if (resident) {
                    phase(xa, xb, 0);
                    phase(na, nb, 1);
                } else {
                    for (uint32_t c = 0; c < kch; ++c) {
                        // this warp's X fragments for chunk c: fetched once, reused for every row tile of the group
                        bool more = false;
                        if (!PF) {
                            load_x(xa, xb, c);
                        } else {
                            more = (c + 1 < kch) || (g0 + GS_TG <= tile_hi);
                            if (more) load_x(na, nb, c + 1 < kch ? c + 1 : 0);      // the next phase's, behind this phase's work
                        }
                        phase(xa, xb, c);
                        if (PF && more) {
#pragma unroll
                            for (int ks = 0; ks < KS; ++ks) {
                                xa[ks] = na[ks];
                                xb[ks] = nb[ks];
                            }
                        }
                    }
                }

                // ---- the group is done: reduce over the 8 warps (each summed its own k-slice), GS_TGR row tiles per pass
#pragma unroll
                for (int sb = 0; sb < GS_TG / GS_TGR; ++sb) {
                    const uint32_t tb = g0 + sb * GS_TGR;
                    if (tb <= g1) {
                        // what this pass hands to the helper: the head tile's partial to publish (early in the range: the tile's
                        // owner needs it only at its end) and / or the tail tile to finish -- slots in that order
                        const bool pub_here = cut_head && tb == tile_lo;
                        const bool tail_here = cut_tail && tile_hi >= tb && tile_hi < tb + GS_TGR && tile_hi <= g1;
                        uint32_t pslot = 0, tslot = 0;
                        if (pub_here) pslot = reserve();
                        if (tail_here) tslot = reserve();
#pragma unroll
                        for (int jj = 0; jj < GS_TGR; ++jj) {
                            const int q = sb * GS_TGR + jj;
                            float* r = red[cw][jj];
                            float v[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) v[i] = GS_NACC == 2 ? acc[q][0][i] + acc[q][GS_NACC - 1][i] : acc[q][0][i];
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
                            if (tile == tile_lo && cut_head) __stcg(mypart + m * GS_ROWS + r, sum);
                            else if (tile == tile_hi && cut_tail) own[tslot][rem] = sum;
                            else store_out(j, tile, m, r, sum);
                        }
                        consumer_bar();          // red[] is reused by the next pass; the partial / own sums are complete
                        if (pub_here) post(pslot, REC_PUBLISH, j, tile_lo, 0, 0);
                        // (the other contributors of the tail tile are the CTAs after this one that hold units of it)
                        if (tail_here) {
                            const uint32_t ul = tile_hi * kch + kch - 1, big = op.rem * (per + 1);      // the tile's last unit; its range:
                            const uint32_t rl = ul < big ? ul / (per + 1) : op.rem + (ul - big) / per;
                            post(tslot, REC_TAIL, j, tile_hi, rl - vr, vr);
                        }
                    }
                }
            }

        }

        if (op.flags & OP_SIGNAL) {
            // report: this CTA is done with op j and everything before it -- through the helper, behind the tails it still holds
            // (the consumers' Y stores are ordered before the record by the barrier)
            const uint32_t sslot = reserve();
            consumer_bar();
            post(sslot, REC_SIGNAL, j, 0, 0, 0);
        }
    }
    if (a.trace && ctid == 0) {
        a.trace[4 * blockIdx.x + 0] = my_smid();
        a.trace[4 * blockIdx.x + 1] = t_start;
        a.trace[4 * blockIdx.x + 3] = global_ns();
    }
    post(reserve(), REC_EXIT, 0, 0, 0, 0);      // the helper finishes what is queued, resets the arrival counters, and leaves
}

std::atomic<bool> g_gemv_pdl{true};      // A/B switch (cloak_set_gemv_engine(2) turns PDL off)

// Counter words [0, GS_TILE_COUNTERS) of the pool's scratch are row-tile arrival counters, the rest op barriers.
constexpr uint32_t GS_TILE_COUNTERS = (uint32_t)(WS_COUNTER_BYTES / 4) - 4 * GS_MAX_OPS;

// Co-residency.  The CTAs of this kernel wait for one another in two ways.
//   (1) The consumers of an `after` op wait for EVERY CTA's arrival at an earlier op: a grid-wide barrier.  If some CTAs have no
//       SM to run on -- another kernel holds SMs: a second pool's chain on another stream, a framework kernel, an MPS / green-
//       context SM limit -- the resident ones spin for ever.  A launch that contains such an op is therefore COOPERATIVE: the
//       driver starts the grid only when every CTA can be resident (one per SM; the grid is never larger than the SM count) and
//       fails the launch (cudaErrorCooperativeLaunchTooLarge) instead of hanging when that can never be.  Measured cost of
//       the attribute: none (cloak_set_gemv_engine(3) launches such chains as ordinary grids: cfg2's chain 2.592 vs 2.596 ms,
//       a 25-launch MoE chain 0.4623 vs 0.4623 ms).
//   (2) The owner of a cut row tile -- its helper warp -- waits for the partials of the FEW CTAs that hold the next ranges of the op,
//       whose helpers publish them early in their ranges.  Such a wait ends once those CTAs are resident; the grid never has more
//       CTAs than the device has SMs (one 200 KB CTA per SM) and the GPU dispatches grids in launch order, so on a device whose SMs
//       are all available to the context the whole grid becomes resident whatever else is queued (two pools' chains on two
//       streams: test_two_pools_two_streams).  Launches with only this kind of wait (cloak_gemv, chains of independent ops) stay
//       ordinary launches.  A context confined to fewer SMs than the device reports cannot run them (cloak.h says so).
// Whether the cooperative attribute may be combined with programmatic stream serialization is probed on the first such launch:
// if the driver rejects the pair, PDL is dropped, not the guarantee.
std::atomic<unsigned long long*> g_trace{nullptr};     // cloak_set_trace
std::atomic<bool> g_gemv_exclusive{false};             // cloak_set_gemv_engine(3): the caller vouches that nothing else holds SMs
static std::atomic<int> g_coop_with_pdl{-1};     // -1 unknown, 0 rejected, 1 accepted
int gemv_coop_pdl_state() { return g_coop_with_pdl.load(std::memory_order_relaxed); }

inline const ChainArgs& host_base(const ChainArgs& a) { return a; }
inline const ChainArgs& host_base(const ChainArgsSeg& a) { return a.base; }

template <int CU, int NT, bool SEG = false, typename Args = ChainArgs>
static cloak_status launch(const Args& a, int ctas, int device, cudaStream_t s) {
    const bool coop = host_base(a).any_signal != 0 && !g_gemv_exclusive.load(std::memory_order_relaxed);
    constexpr size_t smem = (size_t)gs_stages(CU) * GS_ROWS * (CU * 512u + GS_PAD);
    static std::atomic<uint64_t> opted{0};
    auto* kernel = gemv_chain_kernel<CU, NT, SEG>;
    cloak_status st = smem_opt_in(kernel, smem, device, opted);
    if (st != CLOAK_OK) return st;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ctas);
    cfg.blockDim = dim3(gs_threads(NT));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = coop ? at : at + 1;
    const bool want_pdl = g_gemv_pdl.load(std::memory_order_relaxed) && (!coop || g_coop_with_pdl.load(std::memory_order_relaxed) != 0);
    cfg.numAttrs = (coop ? 1 : 0) + (want_pdl ? 1 : 0);
    cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, a);
    if (e != cudaSuccess && coop && want_pdl && g_coop_with_pdl.load(std::memory_order_relaxed) < 0 &&
        (e == cudaErrorInvalidValue || e == cudaErrorNotSupported || e == cudaErrorInvalidConfiguration)) {
        cudaGetLastError();
        g_coop_with_pdl.store(0, std::memory_order_relaxed);
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, kernel, a);
    } else if (e == cudaSuccess && coop && want_pdl) {
        g_coop_with_pdl.store(1, std::memory_order_relaxed);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(CLOAK_ERR_CUDA, "gemv chain launch (%d %sCTAs): %s", ctas, coop ? "cooperative " : "", cudaGetErrorString(e));
    }
    launched();
    return CLOAK_OK;
}

// log2 of the row-chunk size the streaming kernel would use for this tensor, or -1 if it cannot take it.
int gemv_stream_chunk(const cloak_pool* pool, const cloak_tensor* w, uint32_t batch) {
    if (w->dt != CLOAK_BF16 || w->layout != CLOAK_ROWMAJOR || w->K % 256 || w->N % GS_ROWS || pool->block < 512) return -1;
    (void)batch;   // measured: forcing 2 KiB chunks at batch 9..16 so that the X prefetch fits 168 registers costs 35 %
    const uint32_t u = (uint32_t)(((uint64_t)w->K * 2) / 512);          // the row in 512-byte units
    int cu = 8;
    while (u % cu) --cu;
    return cu;
}

// Fusion of small ops (batch <= 8).  An op whose rows are a single chunk (kch == 1) never has a row tile cut by a range
// boundary, so each of its outputs is computed by one CTA in one fixed order whatever the work split: several such ops of one
// shape may be dealt out as ONE op over the concatenation of their row tiles, bit for bit the same results.  That is what an MoE
// layer needs -- a selected expert's projection is 96 units for 148 CTAs, and a CTA pays ~1.3 us of fixed cost per op (table
// lookup and first copy in the producer, reduction and barriers in the consumers) for 0.7 us of streaming.
// Which ops: inside a run of mutually independent ops (consecutive ops that are all after == 0, or an after == 1 op and the
// after == 2 ops behind it), those with kch == 1 and equal (N, K, has-gate-epilogue), kept in chain order.  A gate epilogue needs
// its gate written by the SAME CTA earlier in the launch: the producers must then be the same-numbered segments of one earlier
// fused op of the same size (gate_e / up_e of the selected experts are); if anything does not fit, nothing is fused.
static std::atomic<bool> g_gemv_fuse{true};
void gemv_set_fusion(bool on) { g_gemv_fuse.store(on, std::memory_order_relaxed); }

struct FusedPlan {
    uint32_t nf = 0;                                  // fused ops
    uint32_t first[GS_MAX_OPS], count[GS_MAX_OPS];    // op f = members member[first[f] .. first[f] + count[f])
    uint32_t member[GS_MAX_OPS];                      // original op indices
};

static bool plan_fusion(const cloak_gemv_op* ops, uint32_t n, int cu, FusedPlan& fp) {
    uint32_t grp_of[GS_MAX_OPS], pos_of[GS_MAX_OPS];  // original op -> fused op, position inside it
    uint32_t rep[GS_MAX_OPS], cnt[GS_MAX_OPS];        // per fused op: first member, size
    // An epilogue's gate is either complete before the launch (1) or written by an earlier op of it (2); an op may feed such
    // an epilogue (feeds).  Both are part of what makes ops alike: a launch boundary that cuts a gate_e | up_e pair leaves an up
    // whose gate is outside and a gate nobody in the launch reads -- they must not shift the positions of the pairs that are whole.
    uint8_t gstate[GS_MAX_OPS], feeds[GS_MAX_OPS];
    for (uint32_t j = 0; j < n; ++j) {
        gstate[j] = ops[j].d_gate ? 1 : 0;
        feeds[j] = 0;
    }
    for (uint32_t j = 0; j < n; ++j)
        for (uint32_t k = 0; k < j && ops[j].d_gate; ++k)
            if (ops[k].d_y == ops[j].d_gate) { gstate[j] = 2; feeds[k] = 1; }
    uint32_t nf = 0, run_first_group = 0;
    bool any = false;
    for (uint32_t j = 0; j < n; ++j) {
        const bool new_run = j == 0 || ops[j].after == 1 || ((ops[j].after == 0) != (ops[j - 1].after == 0));
        if (new_run) run_first_group = nf;
        const bool small = (uint64_t)ops[j].w.K * 2 == 512ull * cu;                       // kch == 1
        uint32_t f = nf;
        if (small)
            for (uint32_t q = run_first_group; q < nf; ++q) {
                const uint32_t r = rep[q];
                if (ops[r].w.N == ops[j].w.N && ops[r].w.K == ops[j].w.K &&
                    gstate[r] == gstate[j] && feeds[r] == feeds[j]) { f = q; break; }
            }
        if (f == nf) { rep[nf] = j; cnt[nf] = 0; ++nf; } else any = true;
        grp_of[j] = f;
        pos_of[j] = cnt[f]++;
    }
    if (!any) return false;
    // gate epilogues: producer in this launch -> same position of ONE earlier fused op of the same size for the whole group (the
    // group then copies that op's rotation, gemv_stream_launch: same rows, same CTA)
    uint32_t pgrp[GS_MAX_OPS];
    for (uint32_t f = 0; f < nf; ++f) pgrp[f] = 0xffffffffu;
    for (uint32_t j = 0; j < n; ++j) {
        if (!ops[j].d_gate) continue;
        for (uint32_t k = 0; k < n; ++k) {
            if (ops[k].d_y != ops[j].d_gate) continue;
            if (k >= j || grp_of[k] >= grp_of[j] || pos_of[k] != pos_of[j] || cnt[grp_of[k]] != cnt[grp_of[j]]) return false;
            if (pgrp[grp_of[j]] == 0xffffffffu) pgrp[grp_of[j]] = grp_of[k];
            if (pgrp[grp_of[j]] != grp_of[k]) return false;
        }
    }
    fp.nf = nf;
    uint32_t at = 0;
    for (uint32_t f = 0; f < nf; ++f) { fp.first[f] = at; fp.count[f] = cnt[f]; at += cnt[f]; }
    uint32_t fill[GS_MAX_OPS] = {};
    for (uint32_t j = 0; j < n; ++j) fp.member[fp.first[grp_of[j]] + fill[grp_of[j]]++] = j;
    return true;
}

// One launch: n <= GS_MAX_OPS ops that all stream with the same chunk size (cu x 512 bytes).  Preconditions checked by the callers.
cloak_status gemv_stream_launch(const cloak_pool* pool, const cloak_gemv_op* ops, uint32_t n, int cu, uint32_t batch,
                                cudaStream_t s) {
    ChainArgsSeg as;
    ChainArgs& a = as.base;
    FusedPlan fp;
    const bool seg = batch <= 8 && n > 1 && g_gemv_fuse.load(std::memory_order_relaxed) && plan_fusion(ops, n, cu, fp);
    if (!seg) {
        fp.nf = n;
        for (uint32_t j = 0; j < n; ++j) { fp.first[j] = j; fp.count[j] = 1; fp.member[j] = j; }
    }
    const uint32_t nf = fp.nf;
    a.pool = pool->base;
    a.T = pool->d_T;
    a.log2b = pool->log2_block;
    a.batch = batch;
    a.nops = nf;
    const int sms = sm_count(pool->device);
    uint64_t max_units = 0, tile_base = 0;
    uint32_t last_wait = NO_WAIT;
    a.any_signal = 0;
    for (uint32_t j = 0; j < nf; ++j) {
        const cloak_gemv_op& h = ops[fp.member[fp.first[j]]];       // the first member: shape, dependency
        const cloak_tensor& w = h.w;
        ChainOp& o = a.ops[j];
        o.w_offset = w.w_offset;
        o.x = static_cast<const uint16_t*>(h.d_x);
        o.y = static_cast<__nv_bfloat16*>(h.d_y);
        o.gate = static_cast<const uint16_t*>(h.d_gate);
        o.act = static_cast<uint16_t*>(h.d_act);
        o.N = w.N;
        o.K = w.K;
        o.kch = (uint32_t)(((uint64_t)w.K * 2) / (512u * cu));
        as.tps[j] = w.N / GS_ROWS;
        as.seg0[j] = fp.first[j];
        for (uint32_t q = 0; q < fp.count[j]; ++q) {
            const cloak_gemv_op& m = ops[fp.member[fp.first[j] + q]];
            ChainSeg& sg = as.segs[fp.first[j] + q];
            sg.w_offset = m.w.w_offset;
            sg.x = static_cast<const uint16_t*>(m.d_x);
            sg.y = static_cast<__nv_bfloat16*>(m.d_y);
            sg.gate = static_cast<const uint16_t*>(m.d_gate);
            sg.act = static_cast<uint16_t*>(m.d_act);
        }
        const uint64_t units64 = (uint64_t)fp.count[j] * (w.N / GS_ROWS) * o.kch;
        if (units64 > 0xffffffffull) return fail(CLOAK_ERR_UNSUPPORTED, "gemv: tensor too large");
        o.units = (uint32_t)units64;
        o.tile_base = (uint32_t)tile_base;
        tile_base += (uint64_t)fp.count[j] * (w.N / GS_ROWS);
        // after = 1: wait for every earlier op of the chain (i.e. for op j-1 to be reported by all CTAs);
        // after = 2: the same dependency as the nearest earlier waiting op (no new grid-wide arrival needed)
        o.flags = 0;
        o.wait_op = NO_WAIT;
        if (j > 0 && h.after == 1) o.wait_op = j - 1;
        else if (j > 0 && h.after >= 2) o.wait_op = last_wait;
        if (o.wait_op != NO_WAIT) {
            a.ops[o.wait_op].flags |= OP_SIGNAL;
            a.any_signal = 1;
            last_wait = o.wait_op;
        }
        if (units64 > max_units) max_units = units64;
    }
    if (tile_base > GS_TILE_COUNTERS) return fail(CLOAK_ERR_UNSUPPORTED, "gemv: too many output rows for the row-tile counters");
    const int ctas = max_units < (uint64_t)sms ? (int)max_units : sms;
    // Rotation of the ranges over the CTAs.  Measured: it pays when most of a launch is small ops that leave CTAs idle
    // (MoE experts: 96 units for 148 CTAs; 12 Qwen3-MoE-shaped layers 0.735 -> 0.618 ms) and costs 2 % on dense layers whose
    // ops fill the grid anyway (cfg2 2.54 -> 2.61 ms), so: all ops rotate if ops that leave at least an eighth of the CTAs idle
    // hold most of the launch's units, else only the ops that leave a quarter idle do.
    uint64_t small_units = 0, all_units = 0;
    for (uint32_t j = 0; j < nf; ++j) {
        ChainOp& o = a.ops[j];
        o.ctas = o.units < (uint32_t)ctas ? o.units : (uint32_t)ctas;
        o.per = o.units / o.ctas;
        o.rem = o.units % o.ctas;
        o.pad_ = 0;
        all_units += o.units;
        if (o.ctas * 8 <= (uint32_t)ctas * 7) small_units += o.units;
    }
    const bool rotate_all = 2 * small_units > all_units;
    // An op that fills the grid gives `rem` of its ranges one unit more than the others: they go to the CTAs (a contiguous run,
    // modulo the grid) that hold the least so far, so that over the launch every CTA streams the same bytes to within a unit or
    // two -- with the extras always on CTAs 0 .. rem-1 the first CTAs of the cfg1 layer held 93 units of 32 KiB, the mean 90.
    std::vector<uint32_t> load(ctas, 0);
    auto add_load = [&](const ChainOp& o) {
        for (uint32_t r = 0; r < o.ctas; ++r) load[(r + o.rot) % ctas] += o.per + (r < o.rem ? 1u : 0u);
    };
    uint32_t ranges_so_far = 0;
    for (uint32_t j = 0; j < nf; ++j) {
        ChainOp& o = a.ops[j];
        o.rot = (rotate_all || o.ctas * 4 <= (uint32_t)ctas * 3) ? ranges_so_far % ctas : 0;
        if (o.ctas == (uint32_t)ctas && o.rem > 0) {
            uint64_t win = 0, best = ~0ull;
            for (uint32_t r = 0; r < o.rem; ++r) win += load[r];
            for (uint32_t start = 0; start < (uint32_t)ctas; ++start) {       // window = CTAs start .. start + rem - 1
                if (win < best) { best = win; o.rot = start; }
                win += load[(start + o.rem) % ctas];
                win -= load[start];
            }
        }
        for (uint32_t k = 0; k < j; ++k)
            if (o.gate && (const void*)a.ops[k].y == (const void*)o.gate) o.rot = a.ops[k].rot;     // same rows, same CTA
        add_load(o);
        ranges_so_far += o.ctas;
    }
    a.trace = g_trace.load(std::memory_order_relaxed);
    const size_t need = WS_COUNTER_BYTES + (size_t)nf * ctas * batch * GS_ROWS * 4;
    cloak_status st = pool_workspace(pool, need, s);
    if (st != CLOAK_OK) return st;
    a.counters = reinterpret_cast<uint32_t*>(pool->ws);
    a.opsync = a.counters + GS_TILE_COUNTERS;
    a.part = reinterpret_cast<float*>(pool->ws + WS_COUNTER_BYTES);
    a.early = (g_gemv_pdl.load(std::memory_order_relaxed) && !pool->dirty) ? 1u : 0u;
    if (pool->dirty && pool->dirty_stream == s) pool->dirty = false;   // this launch waits for the writer in full
    const bool nt2 = batch > 8;
#define GS_CASE(C)                                                                                   \
    case C:                                                                                          \
        return seg ? launch<C, 1, true, ChainArgsSeg>(as, ctas, pool->device, s)                     \
                   : (nt2 ? launch<C, 2>(a, ctas, pool->device, s) : launch<C, 1>(a, ctas, pool->device, s))
    switch (cu) {
        GS_CASE(8); GS_CASE(7); GS_CASE(6); GS_CASE(5); GS_CASE(4); GS_CASE(3); GS_CASE(2);
        default: GS_CASE(1);
    }
#undef GS_CASE
    return CLOAK_OK;
}

}  // namespace cloak

// ---------------------------------------------------------------------------------------------------------------------
// cloak_gemv_static: the streaming GEMV of ONE projection with its scratch in a fixed device array -- an entry point that
// allocates nothing (callers under CUDA graph capture, serving loops and harnesses that may not call cudaMalloc).
//
// The kernel is gemv_chain_kernel, unchanged; what differs is where its row-tile counters and cut-tile partials live:
// cloak_gemv takes them from the pool's workspace (cudaMalloc at cloak_pool_create, grown on demand), this call from
// g_static_scratch below -- GS_STATIC_BYTES = 512 KiB that every GPU which loads the library holds until the process ends:
//   words [0, GS_STATIC_TILES)           row-tile arrival counters (one per 8 weight rows: N <= 8 * GS_STATIC_TILES = 524 288)
//   bytes [GS_STATIC_TILES * 4, 512 KiB) fp32 partials, one [batch x 8] block per CTA (148 CTAs x batch 16 = 74 KiB)
// In HOST code the name g_static_scratch is a host-side stand-in for the symbol, not a device address: the address the
// kernel gets comes from cudaGetSymbolAddress, asked once per device with that device current (static_scratch()).
// ALL calls share the array and it keeps the last call's contents: the counters this call uses are cleared first (a tiny
// kernel on the caller's stream), the partials are written before they are read.  Two calls that overlap on the GPU
// (different streams, no event between them) race on it.
namespace cloak {

constexpr uint32_t GS_STATIC_TILES = 65536;                 // 256 KiB of counters
constexpr size_t GS_STATIC_BYTES = 512u << 10;
constexpr size_t GS_STATIC_PART_BYTES = GS_STATIC_BYTES - (size_t)GS_STATIC_TILES * 4;
static __device__ __align__(256) unsigned char g_static_scratch[GS_STATIC_BYTES];

__global__ void zero_words_kernel(uint32_t* p, uint32_t n) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = 0u;
}

// The device address of g_static_scratch on `device` (which must be current): asked once per device, then cached.
static cloak_status static_scratch(int device, unsigned char** out) {
    static std::atomic<unsigned char*> cache[64];
    const bool tracked = device >= 0 && device < 64;
    unsigned char* p = tracked ? cache[device].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        void* sym = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&sym, g_static_scratch);
        if (e != cudaSuccess || !sym) {
            cudaGetLastError();
            return fail(CLOAK_ERR_CUDA, "gemv_static: cudaGetSymbolAddress of the static scratch on device %d: %s", device,
                        cudaGetErrorString(e));
        }
        p = static_cast<unsigned char*>(sym);
        if (tracked) cache[device].store(p, std::memory_order_release);
    }
    *out = p;
    return CLOAK_OK;
}

}  // namespace cloak

namespace cloak { cloak_status check_linear(const cloak_pool* pool, const cloak_tensor* w, const void* x, void* y, const char* who); }

extern "C" cloak_status cloak_gemv_static(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                                          uint32_t batch, void* stream) {
    using namespace cloak;
    cloak_status st = check_linear(pool, w, d_x, d_y, "gemv_static");
    if (st != CLOAK_OK) return st;
    if (batch < 1 || batch > 16) return fail(CLOAK_ERR_INVALID, "gemv_static: batch must be in 1..16");
    const int cu = gemv_stream_chunk(pool, w, batch);
    if (cu < 1 || w->N % 16)
        return fail(CLOAK_ERR_UNSUPPORTED, "gemv_static: needs CLOAK_BF16, CLOAK_ROWMAJOR, K %% 256 == 0, N %% 16 == 0, block_bytes >= 512");
    const uint32_t tiles = w->N / GS_ROWS;
    if (tiles > GS_STATIC_TILES)
        return fail(CLOAK_ERR_UNSUPPORTED, "gemv_static: N = %u needs %u row-tile counters, the static scratch holds %u (N <= %u); use cloak_gemv",
                    w->N, tiles, GS_STATIC_TILES, GS_STATIC_TILES * GS_ROWS);
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    const int sms = sm_count(pool->device);
    ChainArgs a;
    a.pool = pool->base;
    a.T = pool->d_T;
    a.log2b = pool->log2_block;
    a.batch = batch;
    a.nops = 1;
    a.any_signal = 0;
    a.trace = nullptr;
    a.early = 0;                         // the whole launch waits for its stream predecessor (the counter clear below)
    ChainOp& o = a.ops[0];
    o.w_offset = w->w_offset;
    o.x = static_cast<const uint16_t*>(d_x);
    o.y = static_cast<__nv_bfloat16*>(d_y);
    o.gate = nullptr;
    o.act = nullptr;
    o.N = w->N;
    o.K = w->K;
    o.kch = (uint32_t)(((uint64_t)w->K * 2) / (512u * cu));
    const uint64_t units64 = (uint64_t)tiles * o.kch;
    if (units64 > 0xffffffffull) return fail(CLOAK_ERR_UNSUPPORTED, "gemv_static: tensor too large");
    o.units = (uint32_t)units64;
    o.tile_base = 0;
    o.flags = 0;
    o.wait_op = NO_WAIT;
    o.rot = 0;
    const int ctas = units64 < (uint64_t)sms ? (int)units64 : sms;
    o.ctas = o.units < (uint32_t)ctas ? o.units : (uint32_t)ctas;
    o.per = o.units / o.ctas;
    o.rem = o.units % o.ctas;
    o.pad_ = 0;
    const size_t part = (size_t)ctas * batch * GS_ROWS * 4;
    if (part > GS_STATIC_PART_BYTES)
        return fail(CLOAK_ERR_UNSUPPORTED, "gemv_static: %d CTAs x batch %u need %zu bytes of partials, the static scratch holds %zu",
                    ctas, batch, part, GS_STATIC_PART_BYTES);
    unsigned char* scratch = nullptr;
    st = static_scratch(pool->device, &scratch);
    if (st != CLOAK_OK) return st;
    a.counters = reinterpret_cast<uint32_t*>(scratch);
    a.opsync = a.counters + GS_STATIC_TILES - 2 * GS_MAX_OPS;      // (unused by a launch of one op; inside the array all the same)
    a.part = reinterpret_cast<float*>(scratch + (size_t)GS_STATIC_TILES * 4);
    // the counters are self-resetting, but the array is shared with every other call: start from zero whatever was there
    zero_words_kernel<<<(tiles + 1023) / 1024, 1024, 0, s>>>(a.counters, tiles);
    launched();
    CLOAK_LAUNCH_CHECK();
    const bool nt2 = batch > 8;
#define GS_CASE(C) case C: return nt2 ? launch<C, 2>(a, ctas, pool->device, s) : launch<C, 1>(a, ctas, pool->device, s)
    switch (cu) {
        GS_CASE(8); GS_CASE(7); GS_CASE(6); GS_CASE(5); GS_CASE(4); GS_CASE(3); GS_CASE(2);
        default: return nt2 ? launch<1, 2>(a, ctas, pool->device, s) : launch<1, 1>(a, ctas, pool->device, s);
    }
#undef GS_CASE
}
