// cloak_rekey_inplace: periodic re-randomisation of the block layout INSIDE one pool.
//
// Paper: the virtual-to-physical layout is re-drawn every ~1000-1500 iterations with "no additional memory footprint"
// (PAPER.md:207, :271, :283).  S8 (cloak_relayout) re-keys out of place into a second pool; this call re-keys the block
// permutation of a pool in place:      pool[T_B[i] * b + o]  <-  pool[T_A[i] * b + o]      for every block slot i,
// with T_A the table before the call (key A) and T_B the table of `new_key` over the SAME page map (pages are not
// re-mapped: no driver calls, the physical pages stay where they are).  The result equals the oracle's
// relayout(pool, T_A, T_B) bit for bit, zero pad slots included.
//
// Method.  sigma = T_B o T_A^-1 is a permutation of the block slots; its cycles are found on the host (n <= 2^28 table
// entries, O(n)).  A cycle s_0 -> s_1 -> ... -> s_{L-1} -> s_0 ("the block in s_k goes to s_{k+1}") is cut into segments of
// m slots.  Pass 1 saves the first block of every segment into a spare buffer (n/m blocks: the only extra memory, as
// small as one page).  Pass 2 runs every segment backwards -- s_{k} -> s_{k+1} for k = b-1 .. a+1, then spare -> s_{a+1} -- so
// each write lands on a slot whose old block has already moved on or been saved.  Segments are independent: they are
// dealt round-robin to 148 x 4 copy pipelines, each a ring of TMA bulk copies (global -> shared -> global) like the S4 copy
// engine, which executes its list of moves strictly in order.  Traffic: 2 bytes per payload byte, as out of place.
#include <vector>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

constexpr int RK_WARPS = 4;          // independent pipelines per CTA
constexpr int RK_STAGES = 4;
constexpr uint32_t RK_SPARE = 0x80000000u;   // a move endpoint with this bit set is a block of the spare buffer

struct RekeyArgs {
    char* pool;
    char* spare;
    const uint2* moves;              // (src, dst) block indices in execution order, grouped by pipeline
    const uint32_t* pipe_start;      // [npipes + 1] offsets into moves
    uint32_t log2b;
    uint32_t log2c;                  // chunk = min(block, 8 KiB)
};

__global__ void __launch_bounds__(RK_WARPS * 32) rekey_moves_kernel(RekeyArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[RK_WARPS][RK_STAGES];
    if ((threadIdx.x & 31) != 0) return;
    const int w = threadIdx.x >> 5;
    const uint32_t chunk = 1u << a.log2c;
    const uint32_t lc = a.log2b - a.log2c;                    // log2(chunks per block)
    unsigned char* ring = smem + (size_t)w * RK_STAGES * chunk;
#pragma unroll
    for (int s = 0; s < RK_STAGES; ++s) mbar_init(smem_u32(&bars[w][s]), 1);
    fence_barrier_init();

    const uint32_t pipe = blockIdx.x * RK_WARPS + w;
    const uint32_t m0 = a.pipe_start[pipe];
    const uint64_t mine = (uint64_t)(a.pipe_start[pipe + 1] - m0) << lc;      // units = moves x chunks, in order
    auto addr = [&](uint32_t idx, uint64_t c) -> char* {
        return ((idx & RK_SPARE) ? a.spare : a.pool) + ((uint64_t)(idx & ~RK_SPARE) << a.log2b) + (c << a.log2c);
    };
    auto issue_load = [&](uint64_t i) {
        const uint2 mv = __ldg(a.moves + m0 + (i >> lc));
        const int s = (int)(i % RK_STAGES);
        const uint32_t bar = smem_u32(&bars[w][s]);
        mbar_expect_tx(bar, chunk);
        bulk_g2s(smem_u32(ring + (size_t)s * chunk), addr(mv.x, i & ((1ull << lc) - 1)), chunk, bar);
    };
    // Loads run ahead of stores by at most one block: a later move of the same segment reads the slot the earlier move
    // wrote FROM, never the one it wrote TO, and every load is complete (waited for, in order) before any later store.
    const uint64_t pre = mine < RK_STAGES ? mine : RK_STAGES;
    for (uint64_t i = 0; i < pre; ++i) issue_load(i);
    for (uint64_t i = 0; i < mine; ++i) {
        const int s = (int)(i % RK_STAGES);
        mbar_wait(smem_u32(&bars[w][s]), (uint32_t)((i / RK_STAGES) & 1));
        const uint2 mv = __ldg(a.moves + m0 + (i >> lc));
        bulk_s2g(addr(mv.y, i & ((1ull << lc) - 1)), smem_u32(ring + (size_t)s * chunk), chunk);
        bulk_commit();
        if (i >= 1 && i - 1 + RK_STAGES < mine) {
            bulk_wait_read<1>();
            issue_load(i - 1 + RK_STAGES);
        }
    }
    bulk_wait_all();
}

}  // namespace cloak

using namespace cloak;

extern "C" cloak_status cloak_rekey_inplace(cloak_pool* pool, uint64_t new_key, uint64_t spare_bytes, void* stream) {
    if (!pool) return fail(CLOAK_ERR_INVALID, "rekey_inplace: NULL pool");
    if (pool->flags & CLOAK_POOL_IDENTITY) return fail(CLOAK_ERR_INVALID, "rekey_inplace: an identity pool has no key");
    if (pool->log2_block < 4) return fail(CLOAK_ERR_UNSUPPORTED, "rekey_inplace: block_bytes must be >= 16");
    if (pool->rk) return fail(CLOAK_ERR_INVALID, "rekey_inplace: a page re-key of this pool is in progress");
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    const uint32_t n = pool->nslots, b = pool->block, bpp = pool->bpp;

    // ---- new block tables on the device, both block tables on the host
    AsyncBuf new_tables(s), work(s);
    if (cloak_status ast = new_tables.alloc((size_t)2 * n * 4)) return ast;
    uint32_t* d_new = static_cast<uint32_t*>(new_tables.p);    // blockperm_B | blockinv_B
    cloak_status st = keygen_device(new_key, 1ull << 32, n, d_new, d_new + n, s);
    if (st != CLOAK_OK) return st;
    std::vector<uint32_t> inv_a(n), inv_b(n), pageinv(pool->npages);
    CLOAK_CUDA(cudaMemcpyAsync(inv_a.data(), pool->d_blockinv, (size_t)n * 4, cudaMemcpyDeviceToHost, s));
    CLOAK_CUDA(cudaMemcpyAsync(inv_b.data(), d_new + n, (size_t)n * 4, cudaMemcpyDeviceToHost, s));
    CLOAK_CUDA(cudaMemcpyAsync(pageinv.data(), pool->d_pageinv, (size_t)pool->npages * 4, cudaMemcpyDeviceToHost, s));
    CLOAK_CUDA(cudaStreamSynchronize(s));

    // ---- sigma over the slots of the pool's memory: the block in slot_A(i) goes to slot_B(i), i over ALL nslots
    // logical indices (the zero pad blocks move too, so the result is the oracle's relayout, pad slots included)
    // (real pages: the slot's page may sit in either half of the pool's virtual range, see cloak_pool::page_half)
    auto mem_slot = [&](uint32_t v) { return pool->vmm ? v + (uint32_t)pool->page_half[v / bpp] * n : pageinv[v / bpp] * bpp + v % bpp; };
    std::vector<uint32_t> sigma(2 * (size_t)n, 0xffffffffu);          // indexed by memory slot; slots of unmapped halves stay unused
    for (uint32_t i = 0; i < n; ++i) sigma[mem_slot(inv_a[i])] = mem_slot(inv_b[i]);

    // ---- segment length from the spare budget (default: one page)
    uint64_t spare_blocks = (spare_bytes ? spare_bytes : pool->page) / b;
    if (spare_blocks < 1) spare_blocks = 1;
    const int sms = sm_count(pool->device);
    const uint32_t npipes = (uint32_t)sms * RK_WARPS;
    uint32_t m = (uint32_t)((n + spare_blocks - 1) / spare_blocks);
    if (m < 2) m = 2;

    // ---- cycles -> segments -> per-pipeline move lists (pass 1: saves; pass 2: the segments, each in execution order)
    std::vector<uint8_t> seen(2 * (size_t)n, 0);
    std::vector<uint32_t> cyc;
    std::vector<std::vector<uint2>> save(npipes), run(npipes);
    uint32_t nseg = 0;
    for (uint32_t s0 = 0; s0 < 2 * n; ++s0) {
        if (seen[s0] || sigma[s0] == s0 || sigma[s0] == 0xffffffffu) { seen[s0] = 1; continue; }
        cyc.clear();
        for (uint32_t v = s0; !seen[v]; v = sigma[v]) { seen[v] = 1; cyc.push_back(v); }
        const uint32_t L = (uint32_t)cyc.size();
        for (uint32_t a0 = 0; a0 < L; a0 += m, ++nseg) {
            const uint32_t b0 = a0 + m < L ? a0 + m : L;       // segment: cycle positions [a0, b0)
            const uint32_t p = nseg % npipes;
            save[p].push_back(make_uint2(cyc[a0], RK_SPARE | nseg));                 // old block of s_a0 -> spare
            for (uint32_t k = b0 - 1; k > a0; --k) run[p].push_back(make_uint2(cyc[k], cyc[(k + 1) % L]));
            run[p].push_back(make_uint2(RK_SPARE | nseg, cyc[(a0 + 1) % L]));        // saved block -> s_{a0+1}
        }
    }
    if (nseg == 0) return CLOAK_OK;                             // sigma is the identity (same key): nothing moves

    // ---- upload, run the two passes, swap the tables in stream order
    std::vector<uint2> moves;
    std::vector<uint32_t> start(2 * (npipes + 1));
    for (int pass = 0; pass < 2; ++pass) {
        auto& lists = pass ? run : save;
        for (uint32_t p = 0; p < npipes; ++p) {
            start[pass * (npipes + 1) + p] = (uint32_t)moves.size();
            moves.insert(moves.end(), lists[p].begin(), lists[p].end());
        }
        start[pass * (npipes + 1) + npipes] = (uint32_t)moves.size();
    }
    const size_t mv_b = moves.size() * sizeof(uint2), st_b = start.size() * 4, sp_b = (size_t)nseg * b;
    const size_t mv_pad = (mv_b + 255) & ~(size_t)255, st_pad = (st_b + 255) & ~(size_t)255;
    if (cloak_status ast = work.alloc(mv_pad + st_pad + sp_b)) return ast;
    char* d_buf = static_cast<char*>(work.p);
    CLOAK_CUDA(cudaMemcpyAsync(d_buf, moves.data(), mv_b, cudaMemcpyHostToDevice, s));
    CLOAK_CUDA(cudaMemcpyAsync(d_buf + mv_pad, start.data(), st_b, cudaMemcpyHostToDevice, s));
    RekeyArgs a;
    a.pool = pool->base;
    a.spare = d_buf + mv_pad + st_pad;
    a.moves = reinterpret_cast<const uint2*>(d_buf);
    a.log2b = pool->log2_block;
    a.log2c = pool->log2_block < 13 ? pool->log2_block : 13;
    const size_t smem = (size_t)RK_WARPS * RK_STAGES << a.log2c;
    static std::atomic<uint64_t> opted{0};
    if (cloak_status ost = smem_opt_in(rekey_moves_kernel, 200 * 1024, pool->device, opted)) return ost;
    pool->wrote(s);
    for (int pass = 0; pass < 2; ++pass) {
        a.pipe_start = reinterpret_cast<const uint32_t*>(d_buf + mv_pad) + pass * (npipes + 1);
        rekey_moves_kernel<<<sms, RK_WARPS * 32, smem, s>>>(a);
        launched();
    }
    CLOAK_LAUNCH_CHECK();
    CLOAK_CUDA(cudaMemcpyAsync(pool->d_blockperm, d_new, (size_t)2 * n * 4, cudaMemcpyDeviceToDevice, s));   // perm | inv are adjacent
    if (cloak_status bt = launch_build_table(pool, s)) return bt;
    pool->key = new_key;
    // the host lists were copied from pageable memory: the copies above have consumed them when the calls returned
    CLOAK_CUDA(cudaStreamSynchronize(s));
    return CLOAK_OK;
}
