// S5 cloak_permute_mlp_heads (+ the TILE128 storage conversion and the gated-MLP activation glue).
//
// Definition (north_star (b) "rows of W_gate/W_up and columns of W_down, and whole attention
// heads, permuted together"; PAPER.md:11 "intra-layer weight shuffling", :143 "tensor layout"):
//   pi = keygen(key, (4<<32)|layer, inter);  gate'[r,:] = gate[pi[r],:], up'[r,:] = up[pi[r],:], down'[:,r] = down[:,pi[r]]
//   kappa = keygen(key, (5<<32)|layer, n_kv); rho_g = keygen(key, (6<<32)|(layer*n_kv+g), G)
//   eta[g*G+j] = kappa[g]*G + rho_g[j];  k',v' row groups by kappa; q' row groups, o' column groups by eta.
// Bytes move exactly; HBM-bound (1 read + 1 write per byte).
//   rows    : whole-row gather, 16-byte vectors, 4 rows in flight per CTA iteration.
//   columns : source rows stream through a shared-memory ring (one TMA bulk copy per row, several rows in
//             flight), the expanded column map sits in shared memory too, output vectors are assembled from
//             shared memory and stored coalesced; column groups that are whole 16-byte vectors (heads) skip
//             the staging and move vectors directly.
#include <algorithm>
#include "common.cuh"
#include "async.cuh"
#include "philox.cuh"

namespace cloak {

// One CTA: kappa[n_kv] and eta[n_q] of O8 by rank counting in shared memory (n_kv, G <= 1024).
__global__ void __launch_bounds__(1024) head_maps_kernel(uint32_t key_lo, uint32_t key_hi, uint32_t layer, uint32_t n_q,
                                                         uint32_t n_kv, uint32_t* __restrict__ kappa,
                                                         uint32_t* __restrict__ eta) {
    __shared__ uint64_t r[1024];
    __shared__ uint32_t kap[1024];
    const uint32_t t = threadIdx.x;
    const uint32_t G = n_q / n_kv;
    if (t < n_kv) r[t] = philox_key64(t, layer, 5u, key_lo, key_hi);
    __syncthreads();
    if (t < n_kv) {
        uint32_t rank = 0;
        for (uint32_t k = 0; k < n_kv; ++k) rank += (r[k] < r[t]) || (r[k] == r[t] && k < t);
        kap[rank] = t;
        kappa[rank] = t;
    }
    __syncthreads();
    for (uint32_t g = 0; g < n_kv; ++g) {
        if (t < G) r[t] = philox_key64(t, layer * n_kv + g, 6u, key_lo, key_hi);
        __syncthreads();
        if (t < G) {
            uint32_t rank = 0;
            for (uint32_t k = 0; k < G; ++k) rank += (r[k] < r[t]) || (r[k] == r[t] && k < t);
            eta[g * G + rank] = kap[g] * G + t;      // rho_g[rank] = t
        }
        __syncthreads();
    }
}

__device__ __forceinline__ int4 ldg_stream(const void* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// Where a gathered 16-byte vector goes.  PlainDst: a caller-owned tensor.  PoolDst: straight into a pool through its
// block table (the fused load path: permutation and block scatter in ONE pass over the bytes
// instead of two) -- vector index v of the tensor is arena byte off + 16 v, translated like every other access.
// store(row, cv, vpr, x): vector cv of row `row` of a matrix whose rows hold vpr vectors.
struct PlainDst {
    int4* p;
    __device__ __forceinline__ void store(uint64_t row, uint32_t cv, uint32_t vpr, const int4& x) const { p[row * vpr + cv] = x; }
};
// vptr == 0: CLOAK_ROWMAJOR storage.  vptr != 0: CLOAK_TILE128 storage (O11), vptr = vectors per tile row (16 for bf16, 32 for
// f32): the vector belongs to tile (row / 128, cv / vptr), at vector (row % 128) * vptr + cv % vptr inside it -- the storage
// conversion costs an address computation, not a pass over the bytes.
struct PoolDst {
    char* pool;
    const uint32_t* T;
    uint64_t off;
    uint32_t log2b;
    uint32_t vptr;
    __device__ __forceinline__ void store(uint64_t row, uint32_t cv, uint32_t vpr, const int4& x) const {
        uint64_t v = row * vpr + cv;
        if (vptr) {
            const uint64_t tile = (row >> 7) * (vpr / vptr) + cv / vptr;
            v = tile * 128 * vptr + (row & 127) * vptr + cv % vptr;
        }
        const uint64_t a = off + (v << 4);
        const uint32_t slot = __ldg(T + (a >> log2b));
        *reinterpret_cast<int4*>(pool + ((uint64_t)slot << log2b) + (a & ((1ull << log2b) - 1))) = x;
    }
};

// dst row r' <- src row map[r' / seg] * seg + r' % seg;  rows of vpr 16-byte vectors.
constexpr int ROWS_PER_IT = 4;
template <typename Dst>
__global__ void __launch_bounds__(256) gather_rows_kernel(const int4* __restrict__ src, Dst dst,
                                                          const uint32_t* __restrict__ map, uint32_t seg,
                                                          uint32_t nrows, uint32_t vpr) {
    for (uint32_t r0 = blockIdx.x * ROWS_PER_IT; r0 < nrows; r0 += gridDim.x * ROWS_PER_IT) {
        uint32_t srow[ROWS_PER_IT];
#pragma unroll
        for (int k = 0; k < ROWS_PER_IT; ++k) {
            const uint32_t r = r0 + k;
            srow[k] = r >= nrows ? 0u : (map ? __ldg(map + r / seg) * seg + r % seg : r);     // (no map: rows as they are)
        }
        for (uint32_t v = threadIdx.x; v < vpr; v += blockDim.x) {
            int4 x[ROWS_PER_IT];
#pragma unroll
            for (int k = 0; k < ROWS_PER_IT; ++k)
                if (r0 + k < nrows) x[k] = ldg_stream(src + (uint64_t)srow[k] * vpr + v);
#pragma unroll
            for (int k = 0; k < ROWS_PER_IT; ++k)
                if (r0 + k < nrows) dst.store(r0 + k, v, vpr, x[k]);
        }
    }
}

// dst[row, c'] <- src[row, map[c' / seg] * seg + c' % seg], element type E (2 or 4 bytes), column map entries of
// type M (uint16 when ncols <= 65536, else uint32).
// Dynamic shared memory: colmap[ncols] followed by a ring of NS source rows.  One elected thread keeps the ring
// full with one bulk copy (TMA 1-D, mbarrier completion) per row, so the DRAM latency of row r+1.. hides behind the
// shared-memory gather of row r; the gathered vectors go out as coalesced 16-byte stores.
template <typename E, typename M, typename Dst>
__global__ void __launch_bounds__(512) gather_cols_kernel(const E* __restrict__ src, Dst dst,
                                                          const uint32_t* __restrict__ map, uint32_t seg,
                                                          uint32_t nrows, uint32_t ncols, uint32_t ns) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ __align__(8) uint64_t full[8];
    M* colmap = reinterpret_cast<M*>(sm);
    const uint32_t row_bytes = ncols * sizeof(E);
    unsigned char* ring = sm + (((size_t)ncols * sizeof(M) + 127) & ~(size_t)127);
    for (uint32_t c = threadIdx.x; c < ncols; c += blockDim.x) colmap[c] = (M)(__ldg(map + c / seg) * seg + c % seg);
    if (threadIdx.x == 0) {
        for (uint32_t i = 0; i < ns; ++i) mbar_init(smem_u32(&full[i]), 1);
        fence_barrier_init();
    }
    __syncthreads();
    // rows of this CTA: r_k = blockIdx.x + k * gridDim.x
    const uint32_t mine = blockIdx.x < nrows ? (nrows - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto issue = [&](uint32_t k) {
        const uint32_t st = k % ns, bar = smem_u32(&full[st]);
        mbar_expect_tx(bar, row_bytes);
        bulk_g2s(smem_u32(ring + (size_t)st * row_bytes), src + (uint64_t)(blockIdx.x + k * gridDim.x) * ncols, row_bytes, bar);
    };
    if (threadIdx.x == 0)
        for (uint32_t k = 0; k < ns && k < mine; ++k) issue(k);
    constexpr int EPV = 16 / sizeof(E);
    struct alignas(sizeof(M) * EPV) CmVec { M m[EPV]; };      // the EPV map entries of one output vector: one LDS
    const CmVec* cmv = reinterpret_cast<const CmVec*>(colmap);
    const uint32_t vpr = ncols / EPV;
    // Two rows per pass: the map entries are read once (vectorised) for both, which takes the shared-memory
    // instruction count per output vector from 2 x EPV to EPV + 1/2 -- the gather is LDS-bound, not HBM-bound.
    for (uint32_t k = 0; k < mine; k += 2) {
        const bool two = k + 1 < mine;
        const uint32_t sa = k % ns, sb = (k + 1) % ns;
        mbar_wait(smem_u32(&full[sa]), (k / ns) & 1);
        if (two) mbar_wait(smem_u32(&full[sb]), ((k + 1) / ns) & 1);
        const E* ra = reinterpret_cast<const E*>(ring + (size_t)sa * row_bytes);
        const E* rb = reinterpret_cast<const E*>(ring + (size_t)sb * row_bytes);
        const uint64_t rowa = blockIdx.x + (uint64_t)k * gridDim.x, rowb = rowa + gridDim.x;
        for (uint32_t v = threadIdx.x; v < vpr; v += blockDim.x) {
            const CmVec c = cmv[v];
            union { int4 q; E e[EPV]; } oa, ob;
#pragma unroll
            for (int j = 0; j < EPV; ++j) oa.e[j] = ra[c.m[j]];
            dst.store(rowa, v, vpr, oa.q);
            if (two) {
#pragma unroll
                for (int j = 0; j < EPV; ++j) ob.e[j] = rb[c.m[j]];
                dst.store(rowb, v, vpr, ob.q);
            }
        }
        __syncthreads();                                       // every thread is done with both stages
        if (threadIdx.x == 0) {
            if (k + ns < mine) issue(k + ns);
            if (two && k + 1 + ns < mine) issue(k + 1 + ns);
        }
    }
}

// The same for 2-byte elements, organised around what bounds it: shared-memory WAVEFRONTS.  A 2-byte gather from a random
// column is one LDS per element whose 32 lanes collide on the banks (~3.5 wavefronts per instruction): the kernel above spends
// ~30 wavefronts per 512 output bytes and runs at 4.4 TB/s with the DRAM pipe 41 % busy (profiles/r1_ncu_full_gather.md).  Here
// two source rows are first INTERLEAVED element by element into one row of 32-bit pairs (a conflict-free pass of 16-byte loads,
// two PRMTs per word and 16-byte stores), so that one 32-bit LDS at a source column returns that column of BOTH rows: half the
// gather instructions and half the colliding wavefronts per output byte.  Ring of TMA-fetched source rows as above.
template <typename M, typename Dst>
__global__ void __launch_bounds__(1024) gather_cols_pair_kernel(const uint16_t* __restrict__ src, Dst dst,
                                                               const uint32_t* __restrict__ map, uint32_t seg,
                                                               uint32_t nrows, uint32_t ncols, uint32_t ns) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ __align__(8) uint64_t full[8];
    M* colmap = reinterpret_cast<M*>(sm);
    const uint32_t row_bytes = ncols * 2;
    unsigned char* pairs = sm + (((size_t)ncols * sizeof(M) + 127) & ~(size_t)127);      // [ncols] x (row a, row b)
    unsigned char* ring = pairs + 2 * (size_t)row_bytes;
    for (uint32_t c = threadIdx.x; c < ncols; c += blockDim.x) colmap[c] = (M)(__ldg(map + c / seg) * seg + c % seg);
    if (threadIdx.x == 0) {
        for (uint32_t i = 0; i < ns; ++i) mbar_init(smem_u32(&full[i]), 1);
        fence_barrier_init();
    }
    __syncthreads();
    const uint32_t mine = blockIdx.x < nrows ? (nrows - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto issue = [&](uint32_t k) {
        const uint32_t st = k % ns, bar = smem_u32(&full[st]);
        mbar_expect_tx(bar, row_bytes);
        bulk_g2s(smem_u32(ring + (size_t)st * row_bytes), src + (uint64_t)(blockIdx.x + k * gridDim.x) * ncols, row_bytes, bar);
    };
    if (threadIdx.x == 0)
        for (uint32_t k = 0; k < ns && k < mine; ++k) issue(k);
    struct alignas(sizeof(M) * 8) CmVec { M m[8]; };
    const CmVec* cmv = reinterpret_cast<const CmVec*>(colmap);
    const uint32_t vpr = ncols / 8;
    const uint32_t* pw = reinterpret_cast<const uint32_t*>(pairs);
    for (uint32_t k = 0; k < mine; k += 2) {
        const bool two = k + 1 < mine;
        const uint32_t sa = k % ns, sb = (k + 1) % ns;
        mbar_wait(smem_u32(&full[sa]), (k / ns) & 1);
        if (two) mbar_wait(smem_u32(&full[sb]), ((k + 1) / ns) & 1);
        const int4* ra = reinterpret_cast<const int4*>(ring + (size_t)sa * row_bytes);
        const int4* rb = reinterpret_cast<const int4*>(ring + (size_t)(two ? sb : sa) * row_bytes);
        int4* pv = reinterpret_cast<int4*>(pairs);
        for (uint32_t v = threadIdx.x; v < vpr; v += blockDim.x) {          // interleave: pair word c = (a[c], b[c])
            const int4 a = ra[v], b = rb[v];
            pv[2 * v] = make_int4(__byte_perm(a.x, b.x, 0x5410), __byte_perm(a.x, b.x, 0x7632), __byte_perm(a.y, b.y, 0x5410),
                                  __byte_perm(a.y, b.y, 0x7632));
            pv[2 * v + 1] = make_int4(__byte_perm(a.z, b.z, 0x5410), __byte_perm(a.z, b.z, 0x7632), __byte_perm(a.w, b.w, 0x5410),
                                      __byte_perm(a.w, b.w, 0x7632));
        }
        __syncthreads();                                       // pairs complete; both ring stages are free again
        if (threadIdx.x == 0) {
            if (k + ns < mine) issue(k + ns);
            if (two && k + 1 + ns < mine) issue(k + 1 + ns);
        }
        const uint64_t rowa = blockIdx.x + (uint64_t)k * gridDim.x, rowb = rowa + gridDim.x;
        for (uint32_t v = threadIdx.x; v < vpr; v += blockDim.x) {
            const CmVec c = cmv[v];
            uint32_t p[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) p[j] = pw[c.m[j]];
            dst.store(rowa, v, vpr, make_int4(__byte_perm(p[0], p[1], 0x5410), __byte_perm(p[2], p[3], 0x5410),
                                              __byte_perm(p[4], p[5], 0x5410), __byte_perm(p[6], p[7], 0x5410)));
            if (two)
                dst.store(rowb, v, vpr, make_int4(__byte_perm(p[0], p[1], 0x7632), __byte_perm(p[2], p[3], 0x7632),
                                                  __byte_perm(p[4], p[5], 0x7632), __byte_perm(p[6], p[7], 0x7632)));
        }
        __syncthreads();                                       // the pair buffer is rewritten by the next pass
    }
}

// SHORT rows of 2-byte elements, many matrices per launch (the MoE experts' `down`, O8: 128 matrices of [hidden x 768], a row
// is 1.5 KiB -- in the kernel above 96 of 1024 threads would have work).  blockIdx.y = matrix b: source matrix segsrc[b], column
// map map[b*ncols ..], destination matrix b.  A stage is a block of 2*rp CONSECUTIVE source rows -- contiguous in memory, one
// bulk copy -- which are interleaved into rp rows of 32-bit pairs (rows 2p and 2p+1) and gathered as above, all threads busy.
template <typename M>
__global__ void __launch_bounds__(512) gather_cols_short_kernel(const uint16_t* __restrict__ src, int4* __restrict__ dst,
                                                                const uint32_t* __restrict__ map,
                                                                const uint32_t* __restrict__ segsrc, uint32_t nrows,
                                                                uint32_t ncols, uint32_t rp, uint32_t ns) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ __align__(8) uint64_t full[8];
    M* colmap = reinterpret_cast<M*>(sm);
    const uint32_t row_bytes = ncols * 2, vpr = ncols / 8, stage_bytes = 2 * rp * row_bytes;
    unsigned char* pairs = sm + (((size_t)ncols * sizeof(M) + 127) & ~(size_t)127);      // [rp][ncols] x (row 2p, row 2p+1)
    unsigned char* ring = pairs + stage_bytes;
    const uint32_t b = blockIdx.y;
    src += (uint64_t)(segsrc ? __ldg(segsrc + b) : b) * nrows * ncols;
    dst += (uint64_t)b * nrows * vpr;
    map += (uint64_t)b * ncols;
    for (uint32_t c = threadIdx.x; c < ncols; c += blockDim.x) colmap[c] = (M)__ldg(map + c);
    if (threadIdx.x == 0) {
        for (uint32_t i = 0; i < ns; ++i) mbar_init(smem_u32(&full[i]), 1);
        fence_barrier_init();
    }
    __syncthreads();
    const uint32_t nblk = (nrows + 2 * rp - 1) / (2 * rp);
    const uint32_t mine = blockIdx.x < nblk ? (nblk - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto rows_of = [&](uint32_t k) {                           // rows in this CTA's k-th block
        const uint32_t r0 = (blockIdx.x + k * gridDim.x) * 2 * rp;
        return nrows - r0 < 2 * rp ? nrows - r0 : 2 * rp;
    };
    auto issue = [&](uint32_t k) {
        const uint32_t st = k % ns, bar = smem_u32(&full[st]), bytes = rows_of(k) * row_bytes;
        mbar_expect_tx(bar, bytes);
        bulk_g2s(smem_u32(ring + (size_t)st * stage_bytes), src + (uint64_t)(blockIdx.x + k * gridDim.x) * 2 * rp * ncols, bytes, bar);
    };
    if (threadIdx.x == 0)
        for (uint32_t k = 0; k < ns && k < mine; ++k) issue(k);
    struct alignas(sizeof(M) * 8) CmVec { M m[8]; };
    const CmVec* cmv = reinterpret_cast<const CmVec*>(colmap);
    const uint32_t* pw = reinterpret_cast<const uint32_t*>(pairs);
    int4* pv = reinterpret_cast<int4*>(pairs);
    for (uint32_t k = 0; k < mine; ++k) {
        const uint32_t nr = rows_of(k), np = (nr + 1) / 2;
        mbar_wait(smem_u32(&full[k % ns]), (k / ns) & 1);
        const int4* rv = reinterpret_cast<const int4*>(ring + (size_t)(k % ns) * stage_bytes);
        for (uint32_t i = threadIdx.x; i < np * vpr; i += blockDim.x) {      // interleave: pair word (p, c) = (row 2p [c], row 2p+1 [c])
            const uint32_t p = i / vpr, v = i - p * vpr;
            const int4 x = rv[(2 * p) * vpr + v], y = 2 * p + 1 < nr ? rv[(2 * p + 1) * vpr + v] : x;
            pv[(size_t)p * 2 * vpr + 2 * v] = make_int4(__byte_perm(x.x, y.x, 0x5410), __byte_perm(x.x, y.x, 0x7632),
                                                        __byte_perm(x.y, y.y, 0x5410), __byte_perm(x.y, y.y, 0x7632));
            pv[(size_t)p * 2 * vpr + 2 * v + 1] = make_int4(__byte_perm(x.z, y.z, 0x5410), __byte_perm(x.z, y.z, 0x7632),
                                                            __byte_perm(x.w, y.w, 0x5410), __byte_perm(x.w, y.w, 0x7632));
        }
        __syncthreads();                                       // pairs complete; the ring stage is free again
        if (threadIdx.x == 0 && k + ns < mine) issue(k + ns);
        const uint64_t r0 = (uint64_t)(blockIdx.x + k * gridDim.x) * 2 * rp;
        for (uint32_t i = threadIdx.x; i < np * vpr; i += blockDim.x) {
            const uint32_t p = i / vpr, v = i - p * vpr;
            const CmVec c = cmv[v];
            const uint32_t* row = pw + (size_t)p * ncols;
            uint32_t q[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) q[j] = row[c.m[j]];
            dst[(r0 + 2 * p) * vpr + v] = make_int4(__byte_perm(q[0], q[1], 0x5410), __byte_perm(q[2], q[3], 0x5410),
                                                    __byte_perm(q[4], q[5], 0x5410), __byte_perm(q[6], q[7], 0x5410));
            if (2 * p + 1 < nr)
                dst[(r0 + 2 * p + 1) * vpr + v] = make_int4(__byte_perm(q[0], q[1], 0x7632), __byte_perm(q[2], q[3], 0x7632),
                                                            __byte_perm(q[4], q[5], 0x7632), __byte_perm(q[6], q[7], 0x7632));
        }
        __syncthreads();                                       // the pair buffer is rewritten by the next pass
    }
}

// Column groups that are whole 16-byte vectors (seg % (16 / sizeof(E)) == 0, e.g. heads of 128 columns): the gather
// is a vector-level index remap, no staging needed.  vmap[v'] = source vector of destination vector v'.
template <typename Dst>
__global__ void __launch_bounds__(256) gather_colvecs_kernel(const int4* __restrict__ src, Dst dst,
                                                             const uint32_t* __restrict__ map, uint32_t vseg,
                                                             uint32_t nrows, uint32_t vpr) {
    extern __shared__ uint32_t vmap[];
    for (uint32_t v = threadIdx.x; v < vpr; v += blockDim.x) vmap[v] = __ldg(map + v / vseg) * vseg + v % vseg;
    __syncthreads();
    for (uint32_t r0 = blockIdx.x * ROWS_PER_IT; r0 < nrows; r0 += gridDim.x * ROWS_PER_IT) {
        for (uint32_t v = threadIdx.x; v < vpr; v += blockDim.x) {
            const uint32_t sv = vmap[v];
            int4 x[ROWS_PER_IT];
#pragma unroll
            for (int k = 0; k < ROWS_PER_IT; ++k)
                if (r0 + k < nrows) x[k] = ldg_stream(src + (uint64_t)(r0 + k) * vpr + sv);
#pragma unroll
            for (int k = 0; k < ROWS_PER_IT; ++k)
                if (r0 + k < nrows) dst.store(r0 + k, v, vpr, x[k]);
        }
    }
}

// Fallback when a row (+ map) does not fit in shared memory: gather straight from global memory.
template <typename E>
__global__ void __launch_bounds__(256) gather_cols_global_kernel(const E* __restrict__ src, E* __restrict__ dst,
                                                                 const uint32_t* __restrict__ map, uint32_t seg,
                                                                 uint32_t nrows, uint32_t ncols) {
    const uint64_t total = (uint64_t)nrows * ncols;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t r = (uint32_t)(i / ncols), c = (uint32_t)(i % ncols);
        dst[i] = src[(uint64_t)r * ncols + __ldg(map + c / seg) * seg + c % seg];
    }
}

// ROWMAJOR [N, K] -> TILE128 (O11): one CTA per 128 x 128 tile, pure 16-byte index remap.
__global__ void __launch_bounds__(256) tile128_kernel(const int4* __restrict__ src, int4* __restrict__ dst, uint32_t N,
                                                      uint32_t K, uint32_t vptr /* vectors per tile row */) {
    const uint32_t tiles_k = K / 128;
    const uint32_t ntiles = (N / 128) * tiles_k;
    const uint32_t vrow = tiles_k * vptr;                       // vectors per matrix row
    for (uint32_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const uint32_t tn = t / tiles_k, tk = t % tiles_k;
        const int4* s = src + (uint64_t)tn * 128 * vrow + (uint64_t)tk * vptr;
        int4* d = dst + (uint64_t)t * 128 * vptr;
        for (uint32_t v = threadIdx.x; v < 128 * vptr; v += 4 * blockDim.x) {
            int4 x[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t vv = v + k * blockDim.x;
                x[k] = ldg_stream(s + (uint64_t)(vv / vptr) * vrow + vv % vptr);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) d[v + k * blockDim.x] = x[k];
        }
    }
}

__global__ void silu_mul_f32_kernel(const float* __restrict__ g, const float* __restrict__ u, float* __restrict__ o,
                                    uint64_t n) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const float z = g[i];
        o[i] = z / (1.0f + __expf(-z)) * u[i];
    }
}
__global__ void silu_mul_bf16_kernel(const uint16_t* __restrict__ g, const uint16_t* __restrict__ u,
                                     uint16_t* __restrict__ o, uint64_t n) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const float z = __uint_as_float((uint32_t)g[i] << 16), w = __uint_as_float((uint32_t)u[i] << 16);
        const float y = z / (1.0f + __expf(-z)) * w;
        uint32_t b = __float_as_uint(y);
        b += 0x7FFFu + ((b >> 16) & 1u);                       // round to nearest even
        o[i] = (uint16_t)(b >> 16);
    }
}

template <typename Dst>
static cloak_status rows(const void* src, Dst dst, const uint32_t* map, uint32_t seg, uint32_t nrows,
                         uint64_t row_bytes, int sms, cudaStream_t s) {
    uint32_t ctas = (nrows + ROWS_PER_IT - 1) / ROWS_PER_IT;
    const uint32_t cap = (uint32_t)sms * 8;
    if (ctas > cap) ctas = cap;
    gather_rows_kernel<Dst><<<ctas, 256, 0, s>>>((const int4*)src, dst, map, seg, nrows, (uint32_t)(row_bytes / 16));
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

template <typename E, typename M, typename Dst>
static cloak_status cols_ring(const void* src, Dst dst, const uint32_t* map, uint32_t seg, uint32_t nrows, uint32_t ncols,
                              size_t smem, uint32_t ns, int sms, cudaStream_t s) {
    static std::atomic<uint64_t> opted{0};
    auto* kernel = gather_cols_kernel<E, M, Dst>;
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    cloak_status ost = smem_opt_in(kernel, 200 * 1024, dev, opted);
    if (ost != CLOAK_OK) return ost;
    const uint32_t ctas = nrows < (uint32_t)sms ? nrows : (uint32_t)sms;
    gather_cols_kernel<E, M, Dst><<<ctas, 512, smem, s>>>((const E*)src, dst, map, seg, nrows, ncols, ns);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

static std::atomic<bool> g_cols_pairs{true};     // A/B switch (cloak_set_gather_engine)

template <typename M, typename Dst>
static cloak_status cols_pair(const void* src, Dst dst, const uint32_t* map, uint32_t seg, uint32_t nrows, uint32_t ncols,
                              size_t smem, uint32_t ns, int sms, cudaStream_t s) {
    static std::atomic<uint64_t> opted{0};
    auto* kernel = gather_cols_pair_kernel<M, Dst>;
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    if (cloak_status ost = smem_opt_in(kernel, 200 * 1024, dev, opted)) return ost;
    const uint32_t rows_per_cta = 2;
    uint32_t ctas = (nrows + rows_per_cta - 1) / rows_per_cta;
    if (ctas > (uint32_t)sms) ctas = (uint32_t)sms;
    gather_cols_pair_kernel<M, Dst><<<ctas, 1024, smem, s>>>((const uint16_t*)src, dst, map, seg, nrows, ncols, ns);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

// Only a caller-owned tensor can take the element-by-element fallback.
template <typename E>
static cloak_status cols_fallback(const void* src, PlainDst dst, const uint32_t* map, uint32_t seg, uint32_t nrows,
                                  uint32_t ncols, int sms, cudaStream_t s) {
    gather_cols_global_kernel<E><<<sms * 8, 256, 0, s>>>((const E*)src, (E*)dst.p, map, seg, nrows, ncols);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}
template <typename E>
static cloak_status cols_fallback(const void*, PoolDst, const uint32_t*, uint32_t, uint32_t, uint32_t, int, cudaStream_t) {
    return fail(CLOAK_ERR_UNSUPPORTED, "load: a row of this tensor does not fit the shared-memory ring of the column gather");
}

template <typename E, typename Dst>
static cloak_status cols(const void* src, Dst dst, const uint32_t* map, uint32_t seg, uint32_t nrows, uint32_t ncols,
                         int sms, cudaStream_t s) {
    constexpr uint32_t EPV = 16 / sizeof(E);
    const size_t row_bytes = (size_t)ncols * sizeof(E);
    if (seg % EPV == 0 && (size_t)(ncols / EPV) * 4 <= 48 * 1024) {
        const uint32_t vpr = ncols / EPV;
        uint32_t ctas = (nrows + ROWS_PER_IT - 1) / ROWS_PER_IT;
        if (ctas > (uint32_t)sms * 8) ctas = (uint32_t)sms * 8;
        gather_colvecs_kernel<Dst><<<ctas, 256, (size_t)vpr * 4, s>>>((const int4*)src, dst, map, seg / EPV, nrows, vpr);
        launched();
        CLOAK_LAUNCH_CHECK();
        return CLOAK_OK;
    }
    const size_t msz = ncols <= 65536 ? 2 : 4;
    const size_t cm = ((size_t)ncols * msz + 127) & ~(size_t)127;
    const size_t budget = 200 * 1024;
    if (sizeof(E) == 2 && g_cols_pairs.load(std::memory_order_relaxed) && cm + 4 * row_bytes <= budget) {
        // 2-byte elements: the pair-interleaved gather (map + pair buffer of two rows + a ring of at least two source rows)
        uint32_t ns = (uint32_t)((budget - cm - 2 * row_bytes) / row_bytes);
        if (ns > 6) ns = 6;
        const size_t smem = cm + 2 * row_bytes + (size_t)ns * row_bytes;
        return msz == 2 ? cols_pair<uint16_t, Dst>(src, dst, map, seg, nrows, ncols, smem, ns, sms, s)
                        : cols_pair<uint32_t, Dst>(src, dst, map, seg, nrows, ncols, smem, ns, sms, s);
    }
    uint32_t ns = cm < budget ? (uint32_t)((budget - cm) / row_bytes) : 0;
    if (ns > 6) ns = 6;
    if (ns >= 2) {
        const size_t smem = cm + (size_t)ns * row_bytes;
        return msz == 2 ? cols_ring<E, uint16_t, Dst>(src, dst, map, seg, nrows, ncols, smem, ns, sms, s)
                        : cols_ring<E, uint32_t, Dst>(src, dst, map, seg, nrows, ncols, smem, ns, sms, s);
    }
    return cols_fallback<E>(src, dst, map, seg, nrows, ncols, sms, s);
}


// nmat matrices of [nrows x ncols] 2-byte elements with SHORT rows in one launch: dst matrix b <- columns of src matrix
// segsrc[b] gathered by map[b*ncols ..].  Returns CLOAK_ERR_UNSUPPORTED (without setting the error text) if the shape does
// not suit the kernel; the caller then takes the matrix-by-matrix path.
static bool cols_short_fits(uint32_t ncols) { return ncols % 8 == 0 && (size_t)ncols * 2 <= 8192; }
static cloak_status cols_short_batch(const void* src, void* dst, const uint32_t* map, const uint32_t* segsrc, uint32_t nmat,
                                     uint32_t nrows, uint32_t ncols, int sms, cudaStream_t s) {
    const size_t row_bytes = (size_t)ncols * 2;
    uint32_t rp = (uint32_t)(16384 / row_bytes);
    if (rp < 1) rp = 1;
    if (rp > (nrows + 1) / 2) rp = (nrows + 1) / 2;
    const uint32_t ns = 2;
    const size_t msz = ncols <= 65536 ? 2 : 4;
    const size_t cm = ((size_t)ncols * msz + 127) & ~(size_t)127;
    const size_t smem = cm + (size_t)(1 + ns) * 2 * rp * row_bytes;
    static std::atomic<uint64_t> opted2{0}, opted4{0};
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    const uint32_t nblk = (nrows + 2 * rp - 1) / (2 * rp);
    uint32_t gx = ((uint32_t)sms * 2 + nmat - 1) / nmat;      // ~2 CTAs per SM over all matrices
    if (gx > nblk) gx = nblk;
    if (gx < 1) gx = 1;
    if (msz == 2) {
        if (cloak_status ost = smem_opt_in(gather_cols_short_kernel<uint16_t>, 112 * 1024, dev, opted2)) return ost;
        gather_cols_short_kernel<uint16_t><<<dim3(gx, nmat), 512, smem, s>>>((const uint16_t*)src, (int4*)dst, map, segsrc, nrows, ncols, rp, ns);
    } else {
        if (cloak_status ost = smem_opt_in(gather_cols_short_kernel<uint32_t>, 112 * 1024, dev, opted4)) return ost;
        gather_cols_short_kernel<uint32_t><<<dim3(gx, nmat), 512, smem, s>>>((const uint16_t*)src, (int4*)dst, map, segsrc, nrows, ncols, rp, ns);
    }
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

}  // namespace cloak

using namespace cloak;

namespace cloak {

static cloak_status check_shape(const cloak_block_shape* sh, bool mlp, bool heads, const char* who) {
    const uint32_t e = sh->dt == CLOAK_F32 ? 4 : 2;
    const uint32_t epv = 16 / e;
    if (sh->hidden == 0 || sh->hidden % epv) return fail(CLOAK_ERR_ALIGN, "%s: hidden must be a multiple of %u", who, epv);
    if (mlp && (sh->inter == 0 || sh->inter % epv)) return fail(CLOAK_ERR_ALIGN, "%s: inter must be a multiple of %u", who, epv);
    if (heads) {
        if (sh->n_q == 0 || sh->n_kv == 0 || sh->head_dim == 0 || sh->n_q % sh->n_kv)
            return fail(CLOAK_ERR_INVALID, "%s: n_q must be a non-zero multiple of n_kv, head_dim > 0", who);
        if (sh->n_kv > 1024 || sh->n_q / sh->n_kv > 1024) return fail(CLOAK_ERR_UNSUPPORTED, "%s: more than 1024 KV heads or group size", who);
        if ((sh->n_q * sh->head_dim) % epv) return fail(CLOAK_ERR_ALIGN, "%s: n_q*head_dim must be a multiple of %u", who, epv);
    }
    return CLOAK_OK;
}

// A second stream for the head path.  The MLP path (keygen over `inter`, three large gathers) and the head path (head maps,
// four small launch-bound gathers) are independent: forked from the caller's stream and joined back into it with events --
// which stream capture records as graph dependencies -- the small kernels run in the shadow of the large ones.
struct ForkJoin {
    cudaStream_t aux = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr, mid = nullptr;
    bool ok = false;
    bool init() {
        if (ok) return true;
        ok = cudaStreamCreateWithFlags(&aux, cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&fork, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&join, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&mid, cudaEventDisableTiming) == cudaSuccess;
        if (!ok) cudaGetLastError();
        return ok;
    }
};
static ForkJoin& fork_join(int dev) {
    static thread_local ForkJoin fj[16];
    return fj[dev & 15];
}

// The permutation proper.  in[i] (gate, up, down, q, k, v, o) may be NULL to skip a tensor; mk(i) says where tensor i goes.
template <typename MakeDst>
static cloak_status permute_impl(uint64_t key, const cloak_block_shape* sh, const void* const in[7], MakeDst mk, int dev,
                                 cudaStream_t s) {
    const bool mlp = in[0] || in[1] || in[2], heads = in[3] || in[4] || in[5] || in[6];
    const uint32_t e = sh->dt == CLOAK_F32 ? 4 : 2;
    const int sms = sm_count(dev);
    const size_t n_scratch = (size_t)(mlp ? sh->inter : 0) + (heads ? sh->n_kv + sh->n_q : 0);
    AsyncBuf sbuf(s);
    if (cloak_status ast = sbuf.alloc(n_scratch * 4)) return ast;
    uint32_t* scratch = static_cast<uint32_t*>(sbuf.p);
    uint32_t* pi = scratch;
    uint32_t* kappa = scratch + (mlp ? sh->inter : 0);
    uint32_t* eta = kappa + sh->n_kv;
    cloak_status st = CLOAK_OK;
    const uint64_t hrow = (uint64_t)sh->hidden * e;
    // head path on the forked stream when there is an MLP path to overlap with
    ForkJoin& fj = fork_join(dev);
    const bool forked = mlp && heads && fj.init() && cudaEventRecord(fj.fork, s) == cudaSuccess &&
                        cudaStreamWaitEvent(fj.aux, fj.fork, 0) == cudaSuccess;
    cudaStream_t hs = forked ? fj.aux : s;
    if (heads) {
        head_maps_kernel<<<1, 1024, 0, hs>>>((uint32_t)key, (uint32_t)(key >> 32), sh->layer, sh->n_q, sh->n_kv, kappa, eta);
        launched();
        if (cudaGetLastError() != cudaSuccess) st = fail(CLOAK_ERR_CUDA, "permute: head_maps launch failed");
        const uint32_t d = sh->head_dim;
        if (st == CLOAK_OK && in[3]) st = rows(in[3], mk(3), eta, d, sh->n_q * d, hrow, sms, hs);
        if (st == CLOAK_OK && in[4]) st = rows(in[4], mk(4), kappa, d, sh->n_kv * d, hrow, sms, hs);
        if (st == CLOAK_OK && in[5]) st = rows(in[5], mk(5), kappa, d, sh->n_kv * d, hrow, sms, hs);
        if (st == CLOAK_OK && in[6])
            st = e == 4 ? cols<uint32_t>(in[6], mk(6), eta, d, sh->hidden, sh->n_q * d, sms, hs)
                        : cols<uint16_t>(in[6], mk(6), eta, d, sh->hidden, sh->n_q * d, sms, hs);
    }
    if (st == CLOAK_OK && mlp) {
        st = keygen_device(key, (4ull << 32) | sh->layer, sh->inter, pi, nullptr, s);
        // the column gather of `down` is bound by shared memory, not HBM: it too goes to the forked stream (once pi is
        // there), beside the HBM-bound row gathers of gate and up
        cudaStream_t ds = s;
        if (forked && st == CLOAK_OK && in[2] && cudaEventRecord(fj.mid, s) == cudaSuccess &&
            cudaStreamWaitEvent(fj.aux, fj.mid, 0) == cudaSuccess)
            ds = fj.aux;
        if (st == CLOAK_OK && in[2])
            st = e == 4 ? cols<uint32_t>(in[2], mk(2), pi, 1, sh->hidden, sh->inter, sms, ds)
                        : cols<uint16_t>(in[2], mk(2), pi, 1, sh->hidden, sh->inter, sms, ds);
        if (st == CLOAK_OK && in[0]) st = rows(in[0], mk(0), pi, 1, sh->inter, hrow, sms, s);
        if (st == CLOAK_OK && in[1]) st = rows(in[1], mk(1), pi, 1, sh->inter, hrow, sms, s);
    }
    if (forked) cudaEventRecord(fj.join, fj.aux);
    if (forked) cudaStreamWaitEvent(s, fj.join, 0);                // join: everything after this call sees both paths done
    return st;                                                     // (sbuf is freed on s, behind the join)
}

// Zero the rest of the block that holds arena byte `end` (G4: the tail of a tensor's last block is zero).
__global__ void zero_block_tail_kernel(char* pool, const uint32_t* T, uint64_t end, uint32_t log2b) {
    const uint64_t mask = (1ull << log2b) - 1;
    char* p = pool + ((uint64_t)T[end >> log2b] << log2b);
    for (uint64_t o = (end & mask) + threadIdx.x * 16ull; o <= mask; o += blockDim.x * 16ull)
        *reinterpret_cast<int4*>(p + o) = make_int4(0, 0, 0, 0);
}

}  // namespace cloak

extern "C" cloak_status cloak_set_gather_engine(int engine) {
    if (engine < 0 || engine > 1) return fail(CLOAK_ERR_INVALID, "set_gather_engine: 0 (pair-interleaved column gather) or 1 (element gather)");
    g_cols_pairs.store(engine == 0);
    return CLOAK_OK;
}

extern "C" cloak_status cloak_permute_mlp_heads(uint64_t key, const cloak_block_shape* sh, const void* d_gate,
                                                const void* d_up, const void* d_down, const void* d_q, const void* d_k,
                                                const void* d_v, const void* d_o, void* d_gate_o, void* d_up_o,
                                                void* d_down_o, void* d_q_o, void* d_k_o, void* d_v_o, void* d_o_o,
                                                void* stream) {
    if (!sh) return fail(CLOAK_ERR_INVALID, "permute: shape is NULL");
    if (sh->dt != CLOAK_F32 && sh->dt != CLOAK_BF16) return fail(CLOAK_ERR_UNSUPPORTED, "permute: unknown dtype");
    const void* in[7] = {d_gate, d_up, d_down, d_q, d_k, d_v, d_o};
    void* out[7] = {d_gate_o, d_up_o, d_down_o, d_q_o, d_k_o, d_v_o, d_o_o};
    bool any = false, mlp = false, heads = false;
    for (int i = 0; i < 7; ++i) {
        if ((in[i] == nullptr) != (out[i] == nullptr)) return fail(CLOAK_ERR_INVALID, "permute: src/dst %d must both be set or both NULL", i);
        if (in[i]) {
            if (in[i] == out[i]) return fail(CLOAK_ERR_INVALID, "permute: in-place permutation is not supported");
            if (((uintptr_t)in[i] | (uintptr_t)out[i]) & 15) return fail(CLOAK_ERR_ALIGN, "permute: tensor %d not 16-byte aligned", i);
            any = true;
            (i < 3 ? mlp : heads) = true;
        }
    }
    if (!any) return fail(CLOAK_ERR_INVALID, "permute: nothing to do");
    cloak_status st = check_shape(sh, mlp, heads, "permute");
    if (st != CLOAK_OK) return st;
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    return permute_impl(key, sh, in, [&](int i) { return PlainDst{static_cast<int4*>(out[i])}; }, dev, (cudaStream_t)stream);
}

extern "C" cloak_status cloak_load_mlp_heads(uint64_t key, const cloak_block_shape* sh, cloak_pool* pool,
                                             const void* d_gate, const void* d_up, const void* d_down, const void* d_q,
                                             const void* d_k, const void* d_v, const void* d_o, const uint64_t* h_offsets,
                                             void* stream) {
    if (!sh || !pool || !h_offsets) return fail(CLOAK_ERR_INVALID, "load: NULL argument");
    if (sh->dt != CLOAK_F32 && sh->dt != CLOAK_BF16) return fail(CLOAK_ERR_UNSUPPORTED, "load: unknown dtype");
    const void* in[7] = {d_gate, d_up, d_down, d_q, d_k, d_v, d_o};
    bool mlp = false, heads = false;
    for (int i = 0; i < 7; ++i)
        if (in[i]) {
            if ((uintptr_t)in[i] & 15) return fail(CLOAK_ERR_ALIGN, "load: tensor %d not 16-byte aligned", i);
            (i < 3 ? mlp : heads) = true;
        }
    if (!mlp && !heads) return fail(CLOAK_ERR_INVALID, "load: nothing to do");
    cloak_status st = check_shape(sh, mlp, heads, "load");
    if (st != CLOAK_OK) return st;
    const uint64_t e = sh->dt == CLOAK_F32 ? 4 : 2;
    const uint64_t qd = (uint64_t)sh->n_q * sh->head_dim, kvd = (uint64_t)sh->n_kv * sh->head_dim;
    const uint64_t bytes[7] = {(uint64_t)sh->inter * sh->hidden * e, (uint64_t)sh->inter * sh->hidden * e,
                               (uint64_t)sh->hidden * sh->inter * e, qd * sh->hidden * e, kvd * sh->hidden * e,
                               kvd * sh->hidden * e, (uint64_t)sh->hidden * qd * e};
    if (pool->block < 16) return fail(CLOAK_ERR_UNSUPPORTED, "load: block_bytes must be >= 16");
    for (int i = 0; i < 7; ++i)
        if (in[i]) {
            if (h_offsets[i] % pool->block) return fail(CLOAK_ERR_ALIGN, "load: offset %d is not a block multiple", i);
            if (h_offsets[i] + bytes[i] > (uint64_t)pool->nb * pool->block) return fail(CLOAK_ERR_INVALID, "load: tensor %d exceeds the pool's arena", i);
        }
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    pool->wrote(s);
    st = permute_impl(key, sh, in, [&](int i) { return PoolDst{pool->base, pool->d_T, h_offsets[i], pool->log2_block, 0u}; },
                      pool->device, s);
    for (int i = 0; i < 7 && st == CLOAK_OK; ++i)
        if (in[i] && (h_offsets[i] + bytes[i]) % pool->block) {
            zero_block_tail_kernel<<<1, 256, 0, s>>>(pool->base, pool->d_T, h_offsets[i] + bytes[i], pool->log2_block);
            launched();
            CLOAK_LAUNCH_CHECK();
        }
    return st;
}

// NEXT-2 as the survey words it: every tensor of a model -- permuted (S5), laid out (ROWMAJOR or TILE128) and scattered through
// the block table (S4) in ONE pass over its bytes, sourced from wherever the caller holds the checkpoint (device memory, or
// pinned host memory that the kernels read over PCIe themselves: no staging copy), issued in the order the tensors occupy the
// arena, i.e. the keyed tensor order of cloak_arena_plan -- not the model's order (the load is "the only phase
// in which the full set of weight transfers crosses the PCIe bus", so its order is what Tier 1 hides; :217: permutation and
// pages are decided before any weight is transferred).
extern "C" cloak_status cloak_load_tensors(uint64_t key, const cloak_block_shape* sh, cloak_pool* pool,
                                           const cloak_load_item* h_items, uint32_t n, cloak_layout layout, void* stream) {
    if (!sh || !pool || !h_items || n == 0) return fail(CLOAK_ERR_INVALID, "load_tensors: NULL argument or no items");
    if (sh->dt != CLOAK_F32 && sh->dt != CLOAK_BF16) return fail(CLOAK_ERR_UNSUPPORTED, "load_tensors: unknown dtype");
    if (layout != CLOAK_ROWMAJOR && layout != CLOAK_TILE128) return fail(CLOAK_ERR_UNSUPPORTED, "load_tensors: unknown layout");
    if (pool->block < 16) return fail(CLOAK_ERR_UNSUPPORTED, "load_tensors: block_bytes must be >= 16");
    const uint64_t e = sh->dt == CLOAK_F32 ? 4 : 2;
    const uint32_t epv = (uint32_t)(16 / e);
    bool mlp = false, heads = false;
    for (uint32_t i = 0; i < n; ++i) {
        if (h_items[i].role > CLOAK_ROLE_PLAIN) return fail(CLOAK_ERR_INVALID, "load_tensors: item %u: unknown role", i);
        if (h_items[i].role <= CLOAK_ROLE_DOWN) mlp = true;
        else if (h_items[i].role <= CLOAK_ROLE_O) heads = true;
    }
    if (mlp || heads) {
        cloak_status st = check_shape(sh, mlp, heads, "load_tensors");
        if (st != CLOAK_OK) return st;
    }
    const uint64_t qd = (uint64_t)sh->n_q * sh->head_dim, kvd = (uint64_t)sh->n_kv * sh->head_dim;
    struct Item { const void* src; uint64_t off; uint32_t layer, role, N, K; };
    std::vector<Item> items(n);
    std::vector<uint32_t> layers;
    for (uint32_t i = 0; i < n; ++i) {
        const cloak_load_item& it = h_items[i];
        Item x{it.src, it.arena_offset, it.layer, it.role, it.N, it.K};
        switch (it.role) {
            case CLOAK_ROLE_GATE: case CLOAK_ROLE_UP: x.N = sh->inter; x.K = sh->hidden; break;
            case CLOAK_ROLE_DOWN: x.N = sh->hidden; x.K = sh->inter; break;
            case CLOAK_ROLE_Q: x.N = (uint32_t)qd; x.K = sh->hidden; break;
            case CLOAK_ROLE_K: case CLOAK_ROLE_V: x.N = (uint32_t)kvd; x.K = sh->hidden; break;
            case CLOAK_ROLE_O: x.N = sh->hidden; x.K = (uint32_t)qd; break;
            default: break;
        }
        if (!x.src || ((uintptr_t)x.src & 15)) return fail(CLOAK_ERR_ALIGN, "load_tensors: item %u: source NULL or not 16-byte aligned", i);
        if (x.N == 0 || x.K == 0 || x.K % epv) return fail(CLOAK_ERR_ALIGN, "load_tensors: item %u: K must be a non-zero multiple of %u", i, epv);
        if (layout == CLOAK_TILE128 && (x.N % 128 || x.K % 128)) return fail(CLOAK_ERR_ALIGN, "load_tensors: item %u: TILE128 needs N and K multiples of 128", i);
        if (x.off % pool->block) return fail(CLOAK_ERR_ALIGN, "load_tensors: item %u: offset is not a block multiple", i);
        if (x.off + (uint64_t)x.N * x.K * e > (uint64_t)pool->nb * pool->block) return fail(CLOAK_ERR_INVALID, "load_tensors: item %u exceeds the pool's arena", i);
        items[i] = x;
        if (x.role != CLOAK_ROLE_PLAIN && std::find(layers.begin(), layers.end(), x.layer) == layers.end()) layers.push_back(x.layer);
    }
    // the keyed tensor order: ascending arena offset (cloak_arena_plan placed the tensors in keygen(key, TENSOR) order)
    std::sort(items.begin(), items.end(), [](const Item& a, const Item& b) { return a.off < b.off; });
    for (uint32_t i = 1; i < n; ++i)
        if (items[i].off < items[i - 1].off + (uint64_t)items[i - 1].N * items[i - 1].K * e)
            return fail(CLOAK_ERR_INVALID, "load_tensors: items overlap in the arena");
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    const int sms = sm_count(pool->device);
    // the maps of every layer that occurs, once: pi | kappa | eta per layer
    const size_t per_layer = (size_t)(mlp ? sh->inter : 0) + (heads ? sh->n_kv + sh->n_q : 0);
    AsyncBuf sbuf(s);
    uint32_t* scratch = nullptr;
    if (per_layer && !layers.empty()) {
        if (cloak_status ast = sbuf.alloc(per_layer * layers.size() * 4)) return ast;
        scratch = static_cast<uint32_t*>(sbuf.p);
        for (size_t li = 0; li < layers.size(); ++li) {
            uint32_t* pi = scratch + li * per_layer;
            uint32_t* kappa = pi + (mlp ? sh->inter : 0);
            if (mlp)
                if (cloak_status st = keygen_device(key, (4ull << 32) | layers[li], sh->inter, pi, nullptr, s)) return st;
            if (heads) {
                head_maps_kernel<<<1, 1024, 0, s>>>((uint32_t)key, (uint32_t)(key >> 32), layers[li], sh->n_q, sh->n_kv, kappa,
                                                    kappa + sh->n_kv);
                launched();
                CLOAK_LAUNCH_CHECK();
            }
        }
    }
    // Device memory and pinned host memory can be read by the kernels; pageable host memory cannot.  (Bringing pinned host
    // tensors over with the copy engine into a staging buffer first -- 55 GB/s against the 51 GB/s of SM loads across PCIe --
    // was measured, in stream order and overlapped through a second stream, and dropped: 8.57-8.9 ms for the cfg1 layer against
    // 8.57 ms in place; the in-place read needs no buffer and no extra stream.)
    for (uint32_t i = 0; i < n; ++i) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, items[i].src) != cudaSuccess) {
            cudaGetLastError();
            return fail(CLOAK_ERR_INVALID, "load_tensors: cannot classify a source pointer");
        }
        if (at.type == cudaMemoryTypeUnregistered)
            return fail(CLOAK_ERR_INVALID, "load_tensors: a source is pageable host memory: pin it (cudaHostAlloc / cudaHostRegister) or copy it to the device");
    }
    pool->wrote(s);
    const uint32_t vptr = layout == CLOAK_TILE128 ? (uint32_t)(128 * e / 16) : 0u;     // vectors per tile row
    for (const Item& x : items) {
        PoolDst dst{pool->base, pool->d_T, x.off, pool->log2_block, vptr};
        const uint32_t* pi = nullptr;
        const uint32_t *kappa = nullptr, *eta = nullptr;
        if (x.role != CLOAK_ROLE_PLAIN) {
            const size_t li = std::find(layers.begin(), layers.end(), x.layer) - layers.begin();
            pi = scratch + li * per_layer;
            kappa = pi + (mlp ? sh->inter : 0);
            eta = kappa + sh->n_kv;
        }
        const uint64_t row_bytes = (uint64_t)x.K * e;
        const uint32_t d = sh->head_dim;
        cloak_status st = CLOAK_OK;
        switch (x.role) {
            case CLOAK_ROLE_GATE: case CLOAK_ROLE_UP: st = rows(x.src, dst, pi, 1, x.N, row_bytes, sms, s); break;
            case CLOAK_ROLE_Q: st = rows(x.src, dst, eta, d, x.N, row_bytes, sms, s); break;
            case CLOAK_ROLE_K: case CLOAK_ROLE_V: st = rows(x.src, dst, kappa, d, x.N, row_bytes, sms, s); break;
            case CLOAK_ROLE_DOWN:
                st = e == 4 ? cols<uint32_t>(x.src, dst, pi, 1, x.N, x.K, sms, s) : cols<uint16_t>(x.src, dst, pi, 1, x.N, x.K, sms, s);
                break;
            case CLOAK_ROLE_O:
                st = e == 4 ? cols<uint32_t>(x.src, dst, eta, d, x.N, x.K, sms, s) : cols<uint16_t>(x.src, dst, eta, d, x.N, x.K, sms, s);
                break;
            default: st = rows(x.src, dst, nullptr, 1, x.N, row_bytes, sms, s); break;
        }
        if (st != CLOAK_OK) return st;
        const uint64_t end = x.off + (uint64_t)x.N * x.K * e;
        if (end % pool->block) {
            zero_block_tail_kernel<<<1, 256, 0, s>>>(pool->base, pool->d_T, end, pool->log2_block);
            launched();
            CLOAK_LAUNCH_CHECK();
        }
    }
    return CLOAK_OK;
}

extern "C" cloak_status cloak_permute_experts(uint64_t key, const cloak_moe_shape* sh, const void* d_router,
                                              const void* d_gate, const void* d_up, const void* d_down, void* d_router_o,
                                              void* d_gate_o, void* d_up_o, void* d_down_o, void* stream) {
    if (!sh) return fail(CLOAK_ERR_INVALID, "permute_experts: shape is NULL");
    if (sh->dt != CLOAK_F32 && sh->dt != CLOAK_BF16) return fail(CLOAK_ERR_UNSUPPORTED, "permute_experts: unknown dtype");
    const void* in[4] = {d_router, d_gate, d_up, d_down};
    void* out[4] = {d_router_o, d_gate_o, d_up_o, d_down_o};
    for (int i = 0; i < 4; ++i) {
        if (!in[i] || !out[i] || in[i] == out[i]) return fail(CLOAK_ERR_INVALID, "permute_experts: tensor %d NULL or in place", i);
        if (((uintptr_t)in[i] | (uintptr_t)out[i]) & 15) return fail(CLOAK_ERR_ALIGN, "permute_experts: tensor %d not 16-byte aligned", i);
    }
    const uint32_t e = sh->dt == CLOAK_F32 ? 4 : 2, epv = 16 / e;
    const uint32_t E = sh->n_experts, H = sh->hidden, I = sh->inter;
    if (E == 0 || H == 0 || I == 0 || H % epv || I % epv) return fail(CLOAK_ERR_ALIGN, "permute_experts: hidden and inter must be non-zero multiples of %u", epv);
    if (E > 65536) return fail(CLOAK_ERR_UNSUPPORTED, "permute_experts: more than 65536 experts");
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    const int sms = sm_count(dev);
    // eps on the host (to walk the experts) and on the device (to gather the router's rows): the same Philox keygen
    std::vector<uint32_t> eps;
    keygen_host(key, (7ull << 32) | sh->layer, E, eps);
    AsyncBuf sbuf(s);
    if (cloak_status ast = sbuf.alloc(((size_t)E + I) * 4)) return ast;
    uint32_t* scratch = static_cast<uint32_t*>(sbuf.p);
    uint32_t* d_eps = scratch;
    uint32_t* d_pi = scratch + E;
    cloak_status st = keygen_device(key, (7ull << 32) | sh->layer, E, d_eps, nullptr, s);
    const uint64_t hrow = (uint64_t)H * e, emat = (uint64_t)I * H * e;
    if (st == CLOAK_OK) st = rows(d_router, PlainDst{static_cast<int4*>(d_router_o)}, d_eps, 1, E, hrow, sms, s);
    if (st == CLOAK_OK && e == 2 && I <= 4096 && cols_short_fits(I) && (uint64_t)E * I <= 0xffffffffull && E <= 65535) {
        // Batched path (short expert rows: Qwen3-MoE / DeepSeek-style experts): all E neuron permutations in one launch, gate and
        // up as ONE row gather each over the [E*I x H] stack (source row eps[en]*I + pi_eo[j]), down as one column-gather launch
        // over the E matrices: 5 launches per layer instead of ~5 per expert.
        AsyncBuf mbuf(s);
        if (cloak_status ast = mbuf.alloc((size_t)E * I * 8)) return ast;
        uint32_t* rowmap = static_cast<uint32_t*>(mbuf.p);
        uint32_t* colmap = rowmap + (size_t)E * I;
        st = keygen_small_batch(key, 8ull << 32, (uint64_t)sh->layer * E, d_eps, E, I, rowmap, colmap, s);
        if (st == CLOAK_OK) st = rows(d_gate, PlainDst{static_cast<int4*>(d_gate_o)}, rowmap, 1, E * I, hrow, sms, s);
        if (st == CLOAK_OK) st = rows(d_up, PlainDst{static_cast<int4*>(d_up_o)}, rowmap, 1, E * I, hrow, sms, s);
        if (st == CLOAK_OK) st = cols_short_batch(d_down, d_down_o, colmap, d_eps, E, H, I, sms, s);
        return st;
    }
    for (uint32_t en = 0; en < E && st == CLOAK_OK; ++en) {
        const uint32_t eo = eps[en];                               // new expert en is old expert eo, with eo's own pi
        st = keygen_device(key, (8ull << 32) | ((uint64_t)sh->layer * E + eo), I, d_pi, nullptr, s);
        const char* g = (const char*)d_gate + eo * emat;
        const char* u = (const char*)d_up + eo * emat;
        const char* d = (const char*)d_down + eo * emat;
        if (st == CLOAK_OK) st = rows(g, PlainDst{reinterpret_cast<int4*>((char*)d_gate_o + en * emat)}, d_pi, 1, I, hrow, sms, s);
        if (st == CLOAK_OK) st = rows(u, PlainDst{reinterpret_cast<int4*>((char*)d_up_o + en * emat)}, d_pi, 1, I, hrow, sms, s);
        if (st == CLOAK_OK) {
            PlainDst dd{reinterpret_cast<int4*>((char*)d_down_o + en * emat)};
            st = e == 4 ? cols<uint32_t>(d, dd, d_pi, 1, H, I, sms, s) : cols<uint16_t>(d, dd, d_pi, 1, H, I, sms, s);
        }
    }
    return st;
}

extern "C" cloak_status cloak_to_tile128(const void* d_src, void* d_dst, uint32_t N, uint32_t K, cloak_dtype dt,
                                         void* stream) {
    if (!d_src || !d_dst || d_src == d_dst) return fail(CLOAK_ERR_INVALID, "to_tile128: NULL or aliased pointers");
    if (dt != CLOAK_F32 && dt != CLOAK_BF16) return fail(CLOAK_ERR_UNSUPPORTED, "to_tile128: unknown dtype");
    if (N == 0 || K == 0 || N % 128 || K % 128) return fail(CLOAK_ERR_ALIGN, "to_tile128: N and K must be multiples of 128");
    if (((uintptr_t)d_src | (uintptr_t)d_dst) & 15) return fail(CLOAK_ERR_ALIGN, "to_tile128: pointers not 16-byte aligned");
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    const uint32_t ntiles = (N / 128) * (K / 128);
    const uint32_t cap = (uint32_t)sm_count(dev) * 8;
    tile128_kernel<<<ntiles < cap ? ntiles : cap, 256, 0, (cudaStream_t)stream>>>(
        (const int4*)d_src, (int4*)d_dst, N, K, dt == CLOAK_F32 ? 32u : 16u);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

extern "C" cloak_status cloak_silu_mul(const void* d_g, const void* d_u, void* d_out, uint64_t n, cloak_dtype dt,
                                       void* stream) {
    if (!d_g || !d_u || !d_out || n == 0) return fail(CLOAK_ERR_INVALID, "silu_mul: NULL argument or n == 0");
    const unsigned blocks = (unsigned)((n + 255) / 256 < 1184 ? (n + 255) / 256 : 1184);
    if (dt == CLOAK_F32)
        silu_mul_f32_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>((const float*)d_g, (const float*)d_u, (float*)d_out, n);
    else if (dt == CLOAK_BF16)
        silu_mul_bf16_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>((const uint16_t*)d_g, (const uint16_t*)d_u, (uint16_t*)d_out, n);
    else
        return fail(CLOAK_ERR_UNSUPPORTED, "silu_mul: unknown dtype");
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}
