// cloak_pool_layout_report: layout quality of a pool, computed on the GPU.
//
// Paper: its only security-side metric that needs no attacker is contiguity -- "virtual address ranges backed by contiguous
// physical pages": 91.41 % -> 2.38 % (Llama 3.1 8B), 95.57 % -> 1.57 % (Qwen3 14B) (Table 2; the unit is not
// defined there, G12).  Here, for three sequences
//     blocks in the VA view        s(i) = blockinv[i]                                         i < nb
//     blocks in the physical view  s(i) = pageinv[blockinv[i] / bpp] * bpp + blockinv[i] % bpp   (the dump view D)
//     pages                        s(v) = pageinv[v]                                         v < npages
// a RUN is a maximal stretch i, i+1, ..., i+L-1 of logically consecutive items with s(i+1) = s(i) + 1 throughout: what an
// observer who reads memory in that view's order can still stitch together without the key.  Reported per sequence: the
// fraction of neighbours that stayed neighbours (cloak_pool_adjacency's numbers), the number of runs, the longest run, and
// the histogram of run lengths by power of two (bucket k: 2^k <= L < 2^(k+1)).  An identity pool is one run of everything.
//
// Method: start flags (i == 0 or s(i) != s(i-1) + 1) -> exclusive scan (run index of every item; keygen.cu's one-CTA scan:
// this is a report, n <= 2^28) -> start positions scattered by run index -> run length = next start - this start -> histogram.
#include "common.cuh"

namespace cloak {

__global__ void scan_exclusive_kernel(uint32_t* __restrict__ a, uint32_t M);     // keygen.cu

__device__ __forceinline__ uint32_t seq_value(int mode, const uint32_t* __restrict__ blockinv, const uint32_t* __restrict__ pageinv,
                                              uint32_t bpp, uint32_t i) {
    if (mode == 2) return pageinv[i];
    const uint32_t s = blockinv[i];
    return mode == 0 ? s : pageinv[s / bpp] * bpp + s % bpp;
}

// flag[i] = 1 where a run starts; flag[n] = 0 (so that the scan's last entry is the number of runs)
__global__ void run_flags_kernel(int mode, const uint32_t* __restrict__ blockinv, const uint32_t* __restrict__ pageinv, uint32_t bpp,
                                 uint32_t n, uint32_t* __restrict__ flag) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    uint32_t f = 0;
    if (i < n) f = i == 0 || seq_value(mode, blockinv, pageinv, bpp, i) != seq_value(mode, blockinv, pageinv, bpp, i - 1) + 1;
    flag[i] = f;
}
// after the scan: idx[i] = runs that start before i; item i starts a run iff idx[i + 1] != idx[i]
__global__ void run_starts_kernel(const uint32_t* __restrict__ idx, uint32_t n, uint32_t* __restrict__ pos) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && idx[i + 1] != idx[i]) pos[idx[i]] = i;
}
// out: [0] runs, [1] longest, [2] items in runs of length >= 2, [3 + k] runs with 2^k <= length < 2^(k+1)
__global__ void run_hist_kernel(const uint32_t* __restrict__ pos, const uint32_t* __restrict__ idx, uint32_t n,
                                unsigned long long* __restrict__ out) {
    const uint32_t runs = idx[n];
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r == 0) out[0] = runs;
    if (r >= runs) return;
    const uint32_t len = (r + 1 < runs ? pos[r + 1] : n) - pos[r];
    atomicAdd(out + 3 + (31 - __clz(len)), 1ull);
    atomicMax(out + 1, (unsigned long long)len);
    if (len >= 2) atomicAdd(out + 2, (unsigned long long)len);
}

}  // namespace cloak

using namespace cloak;

extern "C" cloak_status cloak_pool_layout_report(const cloak_pool* pool, cloak_layout_report* h_report, void* stream) {
    if (!pool || !h_report) return fail(CLOAK_ERR_INVALID, "pool_layout_report: NULL argument");
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    const uint32_t nmax = pool->nb > pool->npages ? pool->nb : pool->npages;
    AsyncBuf buf(s);
    const size_t words = 2 * ((size_t)nmax + 1);
    constexpr int OUTW = 3 + 32;
    if (cloak_status ast = buf.alloc(words * 4 + 3 * OUTW * 8)) return ast;
    uint32_t* idx = static_cast<uint32_t*>(buf.p);
    uint32_t* pos = idx + nmax + 1;
    unsigned long long* out = reinterpret_cast<unsigned long long*>(static_cast<char*>(buf.p) + ((words * 4 + 7) & ~(size_t)7));
    CLOAK_CUDA(cudaMemsetAsync(out, 0, 3 * OUTW * 8, s));
    for (int mode = 0; mode < 3; ++mode) {
        const uint32_t n = mode == 2 ? pool->npages : pool->nb;
        run_flags_kernel<<<(n + 256) / 256, 256, 0, s>>>(mode, pool->d_blockinv, pool->d_pageinv, pool->bpp, n, idx);
        scan_exclusive_kernel<<<1, 1024, 0, s>>>(idx, n + 1);
        run_starts_kernel<<<(n + 255) / 256, 256, 0, s>>>(idx, n, pos);
        run_hist_kernel<<<(n + 255) / 256, 256, 0, s>>>(pos, idx, n, out + mode * OUTW);
        launched(4);
        CLOAK_LAUNCH_CHECK();
    }
    unsigned long long h[3 * OUTW];
    CLOAK_CUDA(cudaMemcpyAsync(h, out, sizeof(h), cudaMemcpyDeviceToHost, s));
    CLOAK_CUDA(cudaStreamSynchronize(s));
    cloak_run_stats* dst[3] = {&h_report->va_blocks, &h_report->physical_blocks, &h_report->pages};
    for (int mode = 0; mode < 3; ++mode) {
        const uint32_t n = mode == 2 ? pool->npages : pool->nb;
        const unsigned long long* o = h + mode * OUTW;
        cloak_run_stats& r = *dst[mode];
        r.items = n;
        r.runs = o[0];
        r.longest_run = o[1];
        r.items_in_runs_of_2_or_more = o[2];
        // n items in `runs` runs: n - runs neighbour pairs stayed neighbours, of n - 1
        r.adjacent_fraction = n > 1 ? (double)(n - o[0]) / (double)(n - 1) : 0.0;
        for (int k = 0; k < 32; ++k) r.histogram[k] = o[3 + k];
    }
    return CLOAK_OK;
}
