// S1 cloak_keygen: keyed permutation = indices sorted by Philox4x32-10(key, index).
//
// Definition (BASELINE.json north_star; "a random permutation is
// computed" before any page is allocated):  r_i = o0:o1 of Philox(ctr=(i,0,stream_lo,stream_hi),
// key=(key_lo,key_hi)); perm = indices ascending by (r_i, i); inv[perm[j]] = j.
//
// Kernels (all integer, bit-exact by construction):
//   n <= 4096 : one launch.  Keys in shared memory, rank of i = #{k : (r_k,k) < (r_i,i)} by counting.
//   n  > 4096 : philox_keys -> 8 passes of a stable LSD radix sort on 8-bit digits of the 64-bit key
//               with the index as payload (stable + initial index order ascending == tie-break by
//               smaller i) -> inverse scatter.  Each pass: per-tile histogram, one-CTA exclusive
//               scan over [digit][tile], stable scatter with warp match-any ranking.
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

__global__ void philox_keys_kernel(uint32_t n, uint32_t s_lo, uint32_t s_hi, uint32_t k0, uint32_t k1,
                                   uint64_t* __restrict__ keys, uint32_t* __restrict__ idx) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        keys[i] = philox_key64(i, s_lo, s_hi, k0, k1);
        idx[i] = i;
    }
}

constexpr int RADIX_THREADS = 256;
constexpr int RADIX_WARPS = RADIX_THREADS / 32;
constexpr int RADIX_STEPS = 16;                                  // 32-element steps per warp
constexpr int RADIX_TILE = RADIX_THREADS * RADIX_STEPS;          // 4096 elements per CTA

__global__ void __launch_bounds__(RADIX_THREADS) radix_hist_kernel(const uint64_t* __restrict__ keys, uint32_t n,
                                                                   int shift, uint32_t* __restrict__ hist,
                                                                   uint32_t ntiles) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * RADIX_TILE;
#pragma unroll 4
    for (int j = 0; j < RADIX_STEPS; ++j) {
        uint32_t i = base + j * RADIX_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&h[(uint32_t)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[threadIdx.x * ntiles + blockIdx.x] = h[threadIdx.x];
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

__global__ void __launch_bounds__(RADIX_THREADS) radix_scatter_kernel(
    const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ idx_in, uint64_t* __restrict__ keys_out,
    uint32_t* __restrict__ idx_out, uint32_t n, int shift, const uint32_t* __restrict__ offsets, uint32_t ntiles) {
    __shared__ uint32_t cnt[RADIX_WARPS][256];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j = threadIdx.x; j < RADIX_WARPS * 256; j += RADIX_THREADS) (&cnt[0][0])[j] = 0;
    __syncthreads();
    const uint32_t wbase = blockIdx.x * RADIX_TILE + warp * (32 * RADIX_STEPS);
    uint64_t k[RADIX_STEPS];
    uint32_t rank[RADIX_STEPS];
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int j = 0; j < RADIX_STEPS; ++j) {
        const uint32_t i = wbase + j * 32 + lane;     // a warp owns 512 consecutive elements, in order
        const bool valid = i < n;
        k[j] = valid ? keys_in[i] : 0ull;
        const uint32_t d = (uint32_t)(k[j] >> shift) & 255u;
        const uint32_t active = __ballot_sync(0xffffffffu, valid);
        rank[j] = 0;
        // Every lane reads its digit's running count, then the lowest lane of each digit group bumps it:
        // reads and writes are separated by warp barriers, so there is no divergent shuffle.
        uint32_t peers = 0, old = 0;
        if (valid) {
            peers = __match_any_sync(active, d);
            old = cnt[warp][d];
        }
        __syncwarp();
        if (valid) {
            if ((peers & lt) == 0) cnt[warp][d] = old + __popc(peers);
            rank[j] = old + __popc(peers & lt);
        }
        __syncwarp();
    }
    __syncthreads();
    {   // per digit: global base of this tile, then exclusive prefix over the warps (warp order = element order)
        const uint32_t d = threadIdx.x;
        uint32_t run = offsets[d * ntiles + blockIdx.x];
#pragma unroll
        for (int w = 0; w < RADIX_WARPS; ++w) {
            uint32_t c = cnt[w][d];
            cnt[w][d] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < RADIX_STEPS; ++j) {
        const uint32_t i = wbase + j * 32 + lane;
        if (i < n) {
            const uint32_t d = (uint32_t)(k[j] >> shift) & 255u;
            const uint32_t pos = cnt[warp][d] + rank[j];
            if (keys_out) keys_out[pos] = k[j];
            idx_out[pos] = idx_in[i];
        }
    }
}

__global__ void invert_kernel(const uint32_t* __restrict__ perm, uint32_t* __restrict__ inv, uint32_t n) {
    uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) inv[perm[j]] = j;
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
    const uint32_t ntiles = (n + RADIX_TILE - 1) / RADIX_TILE;
    const size_t keys_b = (size_t)n * 8, idx_b = (size_t)n * 4, hist_b = (size_t)256 * ntiles * 4;
    const size_t total = 2 * keys_b + 2 * idx_b + hist_b;
    char* ws = nullptr;
    {   // keep freed workspace cached in the stream-ordered pool instead of returning it to the OS at every sync
        static bool tuned = false;
        if (!tuned) {
            int dev = 0;
            cudaMemPool_t mp;
            if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&mp, dev) == cudaSuccess) {
                uint64_t keep = ~0ull;
                cudaMemPoolSetAttribute(mp, cudaMemPoolAttrReleaseThreshold, &keep);
            }
            cudaGetLastError();
            tuned = true;
        }
    }
    CLOAK_CUDA(cudaMallocAsync((void**)&ws, total, s));
    uint64_t* keys[2] = {(uint64_t*)ws, (uint64_t*)(ws + keys_b)};
    uint32_t* idx[2] = {(uint32_t*)(ws + 2 * keys_b), (uint32_t*)(ws + 2 * keys_b + idx_b)};
    uint32_t* hist = (uint32_t*)(ws + 2 * keys_b + 2 * idx_b);
    philox_keys_kernel<<<(n + 255) / 256, 256, 0, s>>>(n, s_lo, s_hi, k0, k1, keys[0], idx[0]);
    launched();
    CLOAK_LAUNCH_CHECK();
    int cur = 0;
    for (int pass = 0; pass < 8; ++pass) {
        const int shift = pass * 8;
        radix_hist_kernel<<<ntiles, RADIX_THREADS, 0, s>>>(keys[cur], n, shift, hist, ntiles);
        launched();
        scan_exclusive_kernel<<<1, 1024, 0, s>>>(hist, 256 * ntiles);
        launched();
        const bool last = pass == 7;
        uint32_t* idx_dst = (last && d_perm) ? d_perm : idx[cur ^ 1];
        radix_scatter_kernel<<<ntiles, RADIX_THREADS, 0, s>>>(keys[cur], idx[cur], last ? nullptr : keys[cur ^ 1],
                                                              idx_dst, n, shift, hist, ntiles);
        launched();
        CLOAK_LAUNCH_CHECK();
        cur ^= 1;
    }
    if (d_inv) {
        const uint32_t* perm = d_perm ? d_perm : idx[cur];
        invert_kernel<<<(n + 255) / 256, 256, 0, s>>>(perm, d_inv, n);
        launched();
        CLOAK_LAUNCH_CHECK();
    }
    CLOAK_CUDA(cudaFreeAsync(ws, s));
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
