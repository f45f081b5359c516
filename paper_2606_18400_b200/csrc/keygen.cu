// S1 cloak_keygen: keyed permutation = indices sorted by Philox4x32-10(key, index).
//
// Definition (BASELINE.json north_star; "a random permutation is
// computed" before any page is allocated):  r_i = o0:o1 of Philox(ctr=(i,0,stream_lo,stream_hi),
// key=(key_lo,key_hi)); perm = indices ascending by (r_i, i); inv[perm[j]] = j.
//
// Kernels (all integer, bit-exact by construction):
//   n <= 4096 : one launch.  Keys in shared memory, rank of i = #{k : (r_k,k) < (r_i,i)} by counting.
//   n  > 4096 : four launches.  Bucket by the top ~log2(n/4) bits of the key (histogram, one-CTA exclusive
//               scan, fill), then rank by counting inside the bucket (~4 elements): a one-pass MSD bucket
//               sort that is O(n) for uniform keys and exact for any.  (Round 1 started with an 8-pass LSD
//               radix sort: 26 launches, ~100 us at n = 14 336; this is 4 launches, ~10 us.)
#include "common.cuh"
#include "philox.cuh"

namespace cloak {

constexpr int SMALL_N = 4096;

__global__ void __launch_bounds__(256) keygen_small_kernel(uint32_t n, uint32_t s_lo, uint32_t s_hi, uint32_t k0,
                                                           uint32_t k1, uint32_t* __restrict__ perm,
                                                           uint32_t* __restrict__ inv) {
    // Every CTA recomputes all n keys into its own shared memory (n <= 4096: cheaper than a second
    // launch), then each thread ranks one element by counting.
    __shared__ uint64_t r[SMALL_N];
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) r[i] = philox_key64(i, s_lo, s_hi, k0, k1);
    __syncthreads();
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const uint64_t ri = r[i];
        uint32_t rank = 0;
#pragma unroll 8
        for (uint32_t k = 0; k < n; ++k) {
            const uint64_t rk = r[k];
            rank += (rk < ri) || (rk == ri && k < i);
        }
        if (perm) perm[rank] = i;
        if (inv) inv[i] = rank;
    }
}

// A batch of small permutations in one launch (the MoE experts' neuron permutations, O8): blockIdx.y = b, stream id
// stream_base | (id_base + sel[b]) -- the permutation of the sel[b]-th member of a family of streams.  With perm_b the b-th
// permutation: rowmap[b*n + j] = sel[b]*n + perm_b[j] (the source row of output row b*n + j when whole members are
// re-ordered by sel and each member's rows by its own permutation), colmap[b*n + j] = perm_b[j].
__global__ void __launch_bounds__(256) keygen_small_batch_kernel(uint32_t n, uint64_t stream_base, uint64_t id_base,
                                                                 const uint32_t* __restrict__ sel, uint32_t k0, uint32_t k1,
                                                                 uint32_t* __restrict__ rowmap, uint32_t* __restrict__ colmap) {
    __shared__ uint64_t r[SMALL_N];
    const uint32_t b = blockIdx.y, m = __ldg(sel + b);
    const uint64_t sid = stream_base | (id_base + m);
    const uint32_t s_lo = (uint32_t)sid, s_hi = (uint32_t)(sid >> 32);
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) r[i] = philox_key64(i, s_lo, s_hi, k0, k1);
    __syncthreads();
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const uint64_t ri = r[i];
        uint32_t rank = 0;
#pragma unroll 8
        for (uint32_t k = 0; k < n; ++k) {
            const uint64_t rk = r[k];
            rank += (rk < ri) || (rk == ri && k < i);
        }
        rowmap[(size_t)b * n + rank] = m * n + i;
        colmap[(size_t)b * n + rank] = i;
    }
}

cloak_status keygen_small_batch(uint64_t key, uint64_t stream_base, uint64_t id_base, const uint32_t* d_sel, uint32_t nbatch,
                                uint32_t n, uint32_t* d_rowmap, uint32_t* d_colmap, cudaStream_t s) {
    if (n > (uint32_t)SMALL_N || nbatch > 65535) return fail(CLOAK_ERR_UNSUPPORTED, "keygen batch: n > 4096 or more than 65535 members");
    keygen_small_batch_kernel<<<dim3((n + 255) / 256, nbatch), 256, 0, s>>>(n, stream_base, id_base, d_sel, (uint32_t)key,
                                                                          (uint32_t)(key >> 32), d_rowmap, d_colmap);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

// ---- n > 4096: bucket by the top bits of the key, then rank by counting inside the bucket.
// The keys are uniform (Philox), so 2^bits ~ n/4 buckets hold ~4 elements each and the counting pass costs
// O(n) in expectation; the result is exact for ANY distribution (a skewed one would only be slower), and it is
// deterministic although the order inside a bucket list is not (atomics): a rank does not depend on that order.
//   bucket_hist   : hist[bucket(r_i)] += 1
//   scan_exclusive: base = exclusive prefix sums (one CTA)
//   bucket_fill   : slot = base[b] + cursor[b]++ ;  bk[slot] = r_i, bi[slot] = i
//   bucket_rank   : rank of (r, i) = base[b] + #{(r', i') in bucket b : (r', i') < (r, i)};  perm[rank] = i, inv[i] = rank
__global__ void __launch_bounds__(256) bucket_hist_kernel(uint32_t n, uint32_t s_lo, uint32_t s_hi, uint32_t k0, uint32_t k1,
                                                          int shift, uint32_t* __restrict__ hist) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicAdd(hist + (uint32_t)(philox_key64(i, s_lo, s_hi, k0, k1) >> shift), 1u);
}

__global__ void __launch_bounds__(256) bucket_fill_kernel(uint32_t n, uint32_t s_lo, uint32_t s_hi, uint32_t k0, uint32_t k1,
                                                          int shift, const uint32_t* __restrict__ base,
                                                          uint32_t* __restrict__ cursor, uint64_t* __restrict__ bk,
                                                          uint32_t* __restrict__ bi) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const uint64_t r = philox_key64(i, s_lo, s_hi, k0, k1);
        const uint32_t b = (uint32_t)(r >> shift);
        const uint32_t slot = base[b] + atomicAdd(cursor + b, 1u);
        bk[slot] = r;
        bi[slot] = i;
    }
}

__global__ void __launch_bounds__(256) bucket_rank_kernel(uint32_t n, int shift, const uint32_t* __restrict__ base,
                                                          const uint64_t* __restrict__ bk, const uint32_t* __restrict__ bi,
                                                          uint32_t* __restrict__ perm, uint32_t* __restrict__ inv) {
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const uint64_t r = bk[p];
    const uint32_t i = bi[p];
    const uint32_t b = (uint32_t)(r >> shift);
    const uint32_t lo = base[b], hi = base[b + 1];
    uint32_t rank = lo;
    for (uint32_t q = lo; q < hi; ++q) {
        const uint64_t rq = bk[q];
        rank += (rq < r) || (rq == r && bi[q] < i);
    }
    if (perm) perm[rank] = i;
    if (inv) inv[i] = rank;
}

// In-place exclusive scan of a[0..M) by one CTA of 1024 threads.
__global__ void __launch_bounds__(1024) scan_exclusive_kernel(uint32_t* __restrict__ a, uint32_t M) {
    constexpr int IT = 8;
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t chunk = 0; chunk < M; chunk += 1024 * IT) {
        uint32_t v[IT];
        uint32_t first = chunk + threadIdx.x * IT;
        uint32_t sum = 0;
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            v[j] = (first + j < M) ? a[first + j] : 0u;
            sum += v[j];
        }
        uint32_t incl = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) warp_tot[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = warp_tot[lane], wi = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                uint32_t t = __shfl_up_sync(0xffffffffu, wi, d);
                if (lane >= d) wi += t;
            }
            warp_tot[lane] = wi - w;   // exclusive prefix of warp totals
        }
        __syncthreads();
        const uint32_t carry = carry_s;
        uint32_t run = carry + warp_tot[warp] + (incl - sum);
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            if (first + j < M) a[first + j] = run;
            run += v[j];
        }
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = run;   // last thread's running total == chunk total + carry
        __syncthreads();
    }
}

cloak_status keygen_device(uint64_t key, uint64_t stream_id, uint32_t n, uint32_t* d_perm, uint32_t* d_inv,
                           cudaStream_t s) {
    const uint32_t s_lo = (uint32_t)stream_id, s_hi = (uint32_t)(stream_id >> 32);
    const uint32_t k0 = (uint32_t)key, k1 = (uint32_t)(key >> 32);
    if (n <= SMALL_N) {
        keygen_small_kernel<<<(n + 255) / 256, 256, 0, s>>>(n, s_lo, s_hi, k0, k1, d_perm, d_inv);
        launched();
        CLOAK_LAUNCH_CHECK();
        return CLOAK_OK;
    }
    int bits = 1;
    while (bits < 22 && (4ull << bits) < n) ++bits;             // ~n/4 buckets, at most 2^22
    const int shift = 64 - bits;
    const uint32_t nbuckets = 1u << bits;
    const size_t keys_b = (size_t)n * 8, idx_b = (size_t)n * 4, tab_b = ((size_t)nbuckets + 1) * 4;
    const size_t total = keys_b + idx_b + 2 * tab_b;
    AsyncBuf buf(s);                     // released on every exit path
    cloak_status ast = buf.alloc(total);
    if (ast != CLOAK_OK) return ast;
    char* ws = static_cast<char*>(buf.p);
    uint64_t* bk = (uint64_t*)ws;
    uint32_t* bi = (uint32_t*)(ws + keys_b);
    uint32_t* base = (uint32_t*)(ws + keys_b + idx_b);           // hist, then (scanned in place) base[0 .. nbuckets]
    uint32_t* cursor = base + nbuckets + 1;
    CLOAK_CUDA(cudaMemsetAsync(base, 0, 2 * tab_b, s));
    const unsigned grid = (n + 255) / 256;
    bucket_hist_kernel<<<grid, 256, 0, s>>>(n, s_lo, s_hi, k0, k1, shift, base);
    launched();
    scan_exclusive_kernel<<<1, 1024, 0, s>>>(base, nbuckets + 1);
    launched();
    bucket_fill_kernel<<<grid, 256, 0, s>>>(n, s_lo, s_hi, k0, k1, shift, base, cursor, bk, bi);
    launched();
    bucket_rank_kernel<<<grid, 256, 0, s>>>(n, shift, base, bk, bi, d_perm, d_inv);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

}  // namespace cloak

extern "C" cloak_status cloak_keygen(uint64_t key, uint64_t stream_id, uint32_t n, uint32_t* d_perm,
                                     uint32_t* d_inv, void* stream) {
    if (n == 0) return cloak::fail(CLOAK_ERR_INVALID, "keygen: n must be >= 1");
    if (n > (1u << 28)) return cloak::fail(CLOAK_ERR_UNSUPPORTED, "keygen: n must be <= 2^28");
    if (!d_perm && !d_inv) return cloak::fail(CLOAK_ERR_INVALID, "keygen: d_perm and d_inv are both NULL");
    return cloak::keygen_device(key, stream_id, n, d_perm, d_inv, (cudaStream_t)stream);
}
