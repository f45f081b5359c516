// S2 the page pool: geometry, keyed block/page tables, and the VMM mapper (host C++).
//
// Paper: Tier 2 "randomizes the mapping of virtual addresses to physical HBM pages" with the CUDA VMM
// API at 2 MB granularity; "tensor pointers and access semantics remain unchanged" (
// Table 1b :192-201); pages are allocated in permuted order *before* any weight is transferred
// (PAPER.md:217).  Definitions O4-O5 and reading G6 of SURVEY.md 8(c): handle-creation order stands for
// physical order; emulated pages fold the page map into the table.
#include <string.h>
#include <chrono>
#include "common.cuh"

namespace cloak {

__global__ void iota_kernel(uint32_t* a, uint32_t n) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = i;
}

// T[i] = blockinv[i] (real pages)  or  pageinv[blockinv[i] / bpp] * bpp + blockinv[i] % bpp (emulated).
__global__ void build_table_kernel(const uint32_t* __restrict__ blockinv, const uint32_t* __restrict__ pageinv,
                                   const uint32_t* __restrict__ pageoff, uint32_t* __restrict__ T, uint32_t nb, uint32_t bpp,
                                   int vmm) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nb) {
        uint32_t s = blockinv[i];
        T[i] = vmm ? s + pageoff[s / bpp] : pageinv[s / bpp] * bpp + s % bpp;
    }
}
cloak_status launch_build_table(const cloak_pool* p, cudaStream_t s) {
    build_table_kernel<<<(p->nb + 255) / 256, 256, 0, s>>>(p->d_blockinv, p->d_pageinv, p->d_pageoff, p->d_T, p->nb, p->bpp,
                                                           p->vmm ? 1 : 0);
    launched();
    CLOAK_LAUNCH_CHECK();
    return CLOAK_OK;
}

// Layout quality: how many logical neighbours (i, i+1) are still neighbours in the VA view, in the
// physical (dump) view, and how many neighbouring VA pages are backed by neighbouring physical pages.
__global__ void adjacency_kernel(const uint32_t* __restrict__ blockinv, const uint32_t* __restrict__ pageinv, uint32_t nb,
                                 uint32_t bpp, uint32_t npages, unsigned long long* __restrict__ out) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned va = 0, ph = 0, pg = 0;
    if (i + 1 < nb) {
        const uint32_t a = blockinv[i], b = blockinv[i + 1];
        va = b == a + 1;
        const uint32_t da = pageinv[a / bpp] * bpp + a % bpp, db = pageinv[b / bpp] * bpp + b % bpp;
        ph = db == da + 1;
    }
    if (i + 1 < npages) pg = pageinv[i + 1] == pageinv[i] + 1;
    va = __reduce_add_sync(0xffffffffu, va);
    ph = __reduce_add_sync(0xffffffffu, ph);
    pg = __reduce_add_sync(0xffffffffu, pg);
    if ((threadIdx.x & 31) == 0) {
        if (va) atomicAdd(out + 0, (unsigned long long)va);
        if (ph) atomicAdd(out + 1, (unsigned long long)ph);
        if (pg) atomicAdd(out + 2, (unsigned long long)pg);
    }
}

static cloak_status destroy_impl(cloak_pool* p) {
    if (!p) return CLOAK_OK;
    DeviceGuard g(p->device);
    const DriverApi* d = driver();
    cudaDeviceSynchronize();
    if (p->vmm && d) {
        if (p->alias) {
            d->MemUnmap((CUdeviceptr)p->alias, p->bytes());
            d->MemAddressFree((CUdeviceptr)p->alias, p->bytes());
        }
        rekey_pages_abandon(p);
        if (p->base) {
            bool all0 = true;
            for (uint8_t h : p->page_half) all0 = all0 && h == 0;
            if (all0 && p->page_half.size() == p->npages && p->handles.size() >= p->npages) {
                d->MemUnmap((CUdeviceptr)p->base, p->bytes());
            } else {                                               // pages sit in either half (or creation failed half-way)
                for (uint32_t v = 0; v < p->npages && v < p->page_half.size(); ++v)
                    d->MemUnmap((CUdeviceptr)p->page_va(v, p->page_half[v]), p->page);
            }
            d->MemAddressFree((CUdeviceptr)p->base, 2 * p->bytes());
        }
        for (auto h : p->handles) d->MemRelease(h);
    } else if (p->base) {
        cudaFree(p->base);
    }
    if (p->d_tables) cudaFree(p->d_tables);
    if (p->ws) cudaFree(p->ws);
    cudaGetLastError();
    delete p;
    return CLOAK_OK;
}

static cloak_status map_pages(cloak_pool* p, const std::vector<uint32_t>& pageinv) {
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    CUmemAllocationProp prop = {};
    prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
    prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    prop.location.id = p->device;
    auto t0 = std::chrono::steady_clock::now();
    CUdeviceptr va = 0;
    CLOAK_CU(d->MemAddressReserve(&va, 2 * p->bytes(), 0, 0, 0));     // two halves (see cloak_pool::page_half); half 1 starts unmapped
    p->base = (char*)va;
    p->handles.reserve(p->npages);
    auto since = [](std::chrono::steady_clock::time_point a) {
        return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - a).count();
    };
    // Measured on B200 (driver 580), 7 658 pages: cuMemCreate 77 us per page, cuMemMap 1 us, cuMemSetAccess 191 us per page
    // whether called once over the range, per run or per page; 4 / 8 / 16 host threads make none of the phases faster (the
    // driver serialises them) and the creates slower.  So: one thread, one cuMemSetAccess.
    auto t1 = std::chrono::steady_clock::now();
    for (uint32_t i = 0; i < p->npages; ++i) {          // creation order == physical page index (G6)
        CUmemGenericAllocationHandle h;
        CLOAK_CU(d->MemCreate(&h, p->page, &prop, 0));
        p->handles.push_back(h);
    }
    p->map_create_ms = since(t1);
    t1 = std::chrono::steady_clock::now();
    for (uint32_t v = 0; v < p->npages; ++v)             // VA page v is backed by physical page pageinv[v]
        CLOAK_CU(d->MemMap(va + (uint64_t)v * p->page, p->page, 0, p->handles[pageinv[v]], 0));
    p->map_map_ms = since(t1);
    t1 = std::chrono::steady_clock::now();
    CUmemAccessDesc acc = {};
    acc.location = prop.location;
    acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
    CLOAK_CU(d->MemSetAccess(va, p->bytes(), &acc, 1));
    p->map_access_ms = since(t1);
    p->map_ms = since(t0);
    return CLOAK_OK;
}

static cloak_status ensure_alias(cloak_pool* p) {
    if (p->alias) return CLOAK_OK;
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    CUdeviceptr va = 0;
    CLOAK_CU(d->MemAddressReserve(&va, p->bytes(), 0, 0, 0));
    for (uint32_t i = 0; i < p->npages; ++i) {
        CUresult r = d->MemMap(va + (uint64_t)i * p->page, p->page, 0, p->handles[i], 0);
        if (r != CUDA_SUCCESS) {
            if (i) d->MemUnmap(va, (uint64_t)i * p->page);
            d->MemAddressFree(va, p->bytes());
            return fail(CLOAK_ERR_CUDA, "alias cuMemMap: %s", cu_err(r));
        }
    }
    CUmemAccessDesc acc = {};
    acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    acc.location.id = p->device;
    acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
    CLOAK_CU(d->MemSetAccess(va, p->bytes(), &acc, 1));
    p->alias = (char*)va;
    return CLOAK_OK;
}

static cloak_status create_impl(cloak_pool* p) {
    DeviceGuard g(p->device);
    if (!g.ok) return fail(CLOAK_ERR_CUDA, "pool_create: cannot select device %d", p->device);
    const bool identity = p->flags & CLOAK_POOL_IDENTITY;
    size_t gran = 0;
    if (!(p->flags & CLOAK_POOL_PLAIN_ALLOC)) {
        const DriverApi* d = driver();
        if (!d) return CLOAK_ERR_CUDA;
        CUmemAllocationProp prop = {};
        prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
        prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
        prop.location.id = p->device;
        CLOAK_CUDA(cudaFree(0));   // make sure the primary context exists before driver calls
        CLOAK_CU(d->MemGetAllocationGranularity(&gran, &prop, CU_MEM_ALLOC_GRANULARITY_MINIMUM));
        p->vmm = gran != 0 && p->page % gran == 0;
    }
    const size_t ntab = 2 * (size_t)p->nslots + 3 * (size_t)p->npages + p->nb;
    CLOAK_CUDA(cudaMalloc((void**)&p->d_tables, ntab * sizeof(uint32_t)));
    p->d_blockperm = p->d_tables;
    p->d_blockinv = p->d_blockperm + p->nslots;
    p->d_pageperm = p->d_blockinv + p->nslots;
    p->d_pageinv = p->d_pageperm + p->npages;
    p->d_pageoff = p->d_pageinv + p->npages;
    p->d_T = p->d_pageoff + p->npages;

    cudaStream_t s;
    CLOAK_CUDA(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
    cloak_status st = CLOAK_OK;
    auto run = [&]() -> cloak_status {
        if (identity) {
            iota_kernel<<<(p->nslots + 255) / 256, 256, 0, s>>>(p->d_blockperm, p->nslots);
            launched();
            iota_kernel<<<(p->nslots + 255) / 256, 256, 0, s>>>(p->d_blockinv, p->nslots);
            launched();
            iota_kernel<<<(p->npages + 255) / 256, 256, 0, s>>>(p->d_pageperm, p->npages);
            launched();
            iota_kernel<<<(p->npages + 255) / 256, 256, 0, s>>>(p->d_pageinv, p->npages);
            launched();
            CLOAK_LAUNCH_CHECK();
        } else {
            cloak_status e = keygen_device(p->key, 1ull << 32, p->nslots, p->d_blockperm, p->d_blockinv, s);
            if (e != CLOAK_OK) return e;
            e = keygen_device(p->key, 2ull << 32, p->npages, p->d_pageperm, p->d_pageinv, s);
            if (e != CLOAK_OK) return e;
        }
        CLOAK_CUDA(cudaMemsetAsync(p->d_pageoff, 0, (size_t)p->npages * 4, s));       // every page starts in half 0
        cloak_status bt = launch_build_table(p, s);
        if (bt != CLOAK_OK) return bt;
        p->h_pageperm.resize(p->npages);
        p->h_pageinv.resize(p->npages);
        p->page_half.assign(p->npages, 0);
        std::vector<uint32_t>& pageinv = p->h_pageinv;
        CLOAK_CUDA(cudaMemcpyAsync(p->h_pageperm.data(), p->d_pageperm, (size_t)p->npages * 4, cudaMemcpyDeviceToHost, s));
        CLOAK_CUDA(cudaMemcpyAsync(pageinv.data(), p->d_pageinv, (size_t)p->npages * 4, cudaMemcpyDeviceToHost, s));
        CLOAK_CUDA(cudaStreamSynchronize(s));
        if (p->vmm) {
            cloak_status e = map_pages(p, pageinv);
            if (e != CLOAK_OK) return e;
        } else {
            CLOAK_CUDA(cudaMalloc((void**)&p->base, p->bytes()));
        }
        CLOAK_CUDA(cudaMemsetAsync(p->base, 0, p->bytes(), s));
        // scratch of the GEMV / GEMM calls: there from the start, so that no compute call allocates or synchronises
        cloak_status e = pool_workspace(p, WS_DEFAULT_BYTES, s);
        if (e != CLOAK_OK) return e;
        CLOAK_CUDA(cudaStreamSynchronize(s));
        return CLOAK_OK;
    };
    st = run();
    cudaStreamDestroy(s);
    return st;
}

}  // namespace cloak

extern "C" cloak_status cloak_pool_create(int device, uint64_t payload_bytes, uint32_t block_bytes,
                                          uint64_t page_bytes, uint64_t key, uint32_t flags, cloak_pool** out) {
    using namespace cloak;
    if (!out) return fail(CLOAK_ERR_INVALID, "pool_create: out is NULL");
    *out = nullptr;
    if (payload_bytes == 0 || device < 0) return fail(CLOAK_ERR_INVALID, "pool_create: payload_bytes == 0 or bad device");
    if (block_bytes < 16 || (block_bytes & (block_bytes - 1)))
        return fail(CLOAK_ERR_UNSUPPORTED, "pool_create: block_bytes must be a power of two >= 16");
    if (page_bytes == 0 || page_bytes % block_bytes)
        return fail(CLOAK_ERR_ALIGN, "pool_create: page_bytes must be a non-zero multiple of block_bytes");
    if (flags & ~(uint32_t)(CLOAK_POOL_IDENTITY | CLOAK_POOL_PLAIN_ALLOC))
        return fail(CLOAK_ERR_INVALID, "pool_create: unknown flag bits");
    const uint64_t nb = (payload_bytes + block_bytes - 1) / block_bytes;
    const uint64_t bpp = page_bytes / block_bytes;
    const uint64_t npages = (nb + bpp - 1) / bpp;
    const uint64_t nslots = npages * bpp;
    if (nslots > (1ull << 28) || bpp > 0xffffffffull)
        return fail(CLOAK_ERR_UNSUPPORTED, "pool_create: more than 2^28 block slots");
    cloak_pool* p = new (std::nothrow) cloak_pool();
    if (!p) return fail(CLOAK_ERR_OOM, "pool_create: host allocation failed");
    p->device = device;
    p->payload = payload_bytes;
    p->block = block_bytes;
    p->log2_block = 0;
    while ((1u << p->log2_block) < block_bytes) ++p->log2_block;
    p->page = page_bytes;
    p->key = key;
    p->flags = flags;
    p->nb = (uint32_t)nb;
    p->bpp = (uint32_t)bpp;
    p->npages = (uint32_t)npages;
    p->nslots = (uint32_t)nslots;
    cloak_status st = create_impl(p);
    if (st != CLOAK_OK) {
        char keep[512];
        snprintf(keep, sizeof(keep), "%s", cloak_last_error());
        destroy_impl(p);
        set_error("%s", keep);
        return st;
    }
    *out = p;
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_destroy(cloak_pool* pool) {
    if (!pool) return cloak::fail(CLOAK_ERR_INVALID, "pool_destroy: NULL pool");
    return cloak::destroy_impl(pool);
}

extern "C" cloak_status cloak_pool_info(const cloak_pool* pool, void** d_base, const uint32_t** d_table, uint32_t* nb,
                                        uint32_t* nslots, uint32_t* npages, int* is_vmm) {
    if (!pool) return cloak::fail(CLOAK_ERR_INVALID, "pool_info: NULL pool");
    if (d_base) *d_base = pool->base;
    if (d_table) *d_table = pool->d_T;
    if (nb) *nb = pool->nb;
    if (nslots) *nslots = pool->nslots;
    if (npages) *npages = pool->npages;
    if (is_vmm) *is_vmm = pool->vmm ? 1 : 0;
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_tables(const cloak_pool* pool, uint32_t* h_blockperm, uint32_t* h_blockinv,
                                          uint32_t* h_pageperm, uint32_t* h_pageinv) {
    using namespace cloak;
    if (!pool) return fail(CLOAK_ERR_INVALID, "pool_tables: NULL pool");
    DeviceGuard g(pool->device);
    if (h_blockperm) CLOAK_CUDA(cudaMemcpy(h_blockperm, pool->d_blockperm, (size_t)pool->nslots * 4, cudaMemcpyDeviceToHost));
    if (h_blockinv) CLOAK_CUDA(cudaMemcpy(h_blockinv, pool->d_blockinv, (size_t)pool->nslots * 4, cudaMemcpyDeviceToHost));
    // the page map in force (host copies: a finished page re-key publishes them at once, the device copies in stream order)
    if (h_pageperm) memcpy(h_pageperm, pool->h_pageperm.data(), (size_t)pool->npages * 4);
    if (h_pageinv) memcpy(h_pageinv, pool->h_pageinv.data(), (size_t)pool->npages * 4);
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_dump(const cloak_pool* pool, void* d_out, void* stream) {
    using namespace cloak;
    if (!pool || !d_out) return fail(CLOAK_ERR_INVALID, "pool_dump: NULL argument");
    DeviceGuard g(pool->device);
    const char* src = pool->base;
    if (pool->vmm) {
        cloak_status st = ensure_alias(const_cast<cloak_pool*>(pool));
        if (st != CLOAK_OK) return st;
        src = pool->alias;
    }
    CLOAK_CUDA(cudaMemcpyAsync(d_out, src, pool->bytes(), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_adjacency(const cloak_pool* pool, double* va_blocks, double* physical_blocks, double* pages,
                                             void* stream) {
    using namespace cloak;
    if (!pool) return fail(CLOAK_ERR_INVALID, "pool_adjacency: NULL pool");
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    AsyncBuf buf(s);
    if (cloak_status ast = buf.alloc(3 * sizeof(unsigned long long))) return ast;
    unsigned long long* d = static_cast<unsigned long long*>(buf.p);
    CLOAK_CUDA(cudaMemsetAsync(d, 0, 3 * sizeof(unsigned long long), s));
    const uint32_t n = pool->nb > pool->npages ? pool->nb : pool->npages;
    adjacency_kernel<<<(n + 255) / 256, 256, 0, s>>>(pool->d_blockinv, pool->d_pageinv, pool->nb, pool->bpp, pool->npages, d);
    launched();
    CLOAK_LAUNCH_CHECK();
    unsigned long long h[3] = {0, 0, 0};
    CLOAK_CUDA(cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, s));
    CLOAK_CUDA(cudaStreamSynchronize(s));
    if (va_blocks) *va_blocks = pool->nb > 1 ? (double)h[0] / (pool->nb - 1) : 0.0;
    if (physical_blocks) *physical_blocks = pool->nb > 1 ? (double)h[1] / (pool->nb - 1) : 0.0;
    if (pages) *pages = pool->npages > 1 ? (double)h[2] / (pool->npages - 1) : 0.0;
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_reserve_workspace(cloak_pool* pool, uint64_t bytes) {
    using namespace cloak;
    if (!pool) return fail(CLOAK_ERR_INVALID, "pool_reserve_workspace: NULL pool");
    if (pool->ws_bytes >= bytes) return CLOAK_OK;
    DeviceGuard g(pool->device);
    CLOAK_CUDA(cudaDeviceSynchronize());                 // nothing in flight holds the old scratch
    cloak_status st = pool_workspace(pool, bytes, nullptr);
    if (st != CLOAK_OK) return st;
    CLOAK_CUDA(cudaDeviceSynchronize());                 // the new counters are zero before any stream can use them
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_map_phases(const cloak_pool* pool, double* create_ms, double* map_ms, double* access_ms) {
    if (!pool) return cloak::fail(CLOAK_ERR_INVALID, "pool_map_phases: NULL pool");
    if (create_ms) *create_ms = pool->map_create_ms;
    if (map_ms) *map_ms = pool->map_map_ms;
    if (access_ms) *access_ms = pool->map_access_ms;
    return CLOAK_OK;
}

extern "C" cloak_status cloak_pool_map_ms(const cloak_pool* pool, double* ms) {
    if (!pool || !ms) return cloak::fail(CLOAK_ERR_INVALID, "pool_map_ms: NULL argument");
    *ms = pool->map_ms;
    return CLOAK_OK;
}
