// cloak_rekey_pages_*: periodic re-randomisation of the PHYSICAL PAGE MAP of a pool under live decode.
//
// Paper: Tier 2 "At initialization and then periodically randomizes the mapping of virtual addresses to physical HBM pages"
// (PAPER.md:165); "periodic randomization ... using CUDA VMM APIs ... tensor pointers and access semantics remain unchanged ...
// no additional memory footprint ... The only overhead arises from synchronization points needed to safely remap pages"
// (PAPER.md:205-207); cadence once per 1000 (text, :207) or 1500 (Fig 7, :283) iterations, < 2 % (:271).
//
// Definition (oracle/pool.py rekey_pages).  (pageperm', pageinv') = keygen(new_key, PAGE, npages).  The VA view V -- and with
// it the block table's logical content and every kernel's result -- is unchanged; VA page v is afterwards backed by physical
// page pageinv'[v] (physical index = handle-creation order, G6), i.e. the dump view becomes
//     D'[pageinv'[v] * P + o] = V[v * P + o] = D[pageinv[v] * P + o].
//
// Method: page-at-a-time moves through spare physical pages, WITHOUT stopping the reader.
//   * The pool's virtual range has two halves (cloak_pool::page_half).  To move VA page v from its physical page A to a free
//     physical page F:   (1) host: cuMemMap F at v's address in the OTHER half + cuMemSetAccess -- nobody reads that address
//     yet;  (2) stream: copy the 2 MiB page from the current half to the other one, then switch the table entries of the
//     page's blocks (and d_pageoff[v]) to the other half -- kernels launched before the switch read the old address, kernels
//     launched after it the new one, both hold the same bytes;  (3) once an event recorded behind the switch has completed:
//     host: cuMemUnmap the old address; A is free.  CUDA graphs of decode chains stay valid: they carry the table's
//     address, not its contents.
//   * Which page moves where: the permutation "the content of physical page h goes to physical page pageinv'[pageperm[h]]"
//     is followed cycle by cycle.  A cycle starts by moving some page into a SPARE physical page (cuMemCreate'd by _begin,
//     released when the re-key is finished: the only extra memory, `spare_pages` x 2 MiB); that frees a physical page, the
//     VA page that wants it moves in, which frees the next, ... until the page parked in the spare goes home.  With k spares
//     k cycles are in flight at once.
//   * cloak_rekey_pages_step is non-blocking and is meant to be called between decode steps: it retires the moves whose event
//     has completed (unmap) and issues up to max_moves new ones (map + two small launches).  Driver time is ~0.25-0.45 ms
//     per page on B200 (cuMemSetAccess dominates) and runs on the calling thread while the GPU works on what was launched before.
#include <algorithm>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

struct PageMove {
    uint32_t v;                  // VA page
    uint32_t from, to;           // physical page (handle index) it leaves / enters
    uint8_t old_half;
    cudaEvent_t done;            // recorded behind the table switch
};

struct RekeyPages {
    uint64_t new_key = 0;
    uint32_t nspare = 0;
    std::vector<uint32_t> tgt;        // tgt[v]  = pageinv'[v]: the physical page VA page v must end on
    std::vector<uint32_t> want;       // want[h] = pageperm'[h]: the VA page that must end on physical page h
    std::vector<uint32_t> cur;        // cur[v]  = physical page backing v now (>= npages: a spare)
    std::vector<uint8_t> moving;      // v has a move in flight
    std::vector<uint32_t> free_pages; // physical pages (handle indices) that are mapped nowhere
    std::vector<PageMove> inflight;
    std::vector<cudaEvent_t> events;  // recycled
    uint32_t scan = 0;                // where the search for the next cycle start resumes
    uint32_t todo = 0;                // VA pages not yet on their target (in flight or not)
    uint32_t moves_issued = 0;
};

constexpr int PM_MAX = 16;            // page moves per launch pair
struct PageMoveArgs {
    const char* src[PM_MAX];
    char* dst[PM_MAX];
    uint32_t v[PM_MAX];
    uint32_t newoff[PM_MAX];          // 0 or nslots: the half the page lives in afterwards
    uint32_t n;
    uint32_t log2c;                   // copy chunk (8 KiB)
    uint32_t units_per_page;
};

constexpr int PM_WARPS = 4, PM_STAGES = 4;
// The copy engine's pipelines (copy.cu) over a handful of whole pages: unit u = chunk (u % units_per_page) of move u / units_per_page.
__global__ void __launch_bounds__(PM_WARPS * 32) page_copy_kernel(const __grid_constant__ PageMoveArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t bars[PM_WARPS][PM_STAGES];
    if ((threadIdx.x & 31) != 0) return;
    const int w = threadIdx.x >> 5;
    const uint32_t chunk = 1u << a.log2c;
    unsigned char* ring = smem + (size_t)w * PM_STAGES * chunk;
#pragma unroll
    for (int s = 0; s < PM_STAGES; ++s) mbar_init(smem_u32(&bars[w][s]), 1);
    fence_barrier_init();
    const uint32_t total = a.n * a.units_per_page;
    const uint32_t npipes = gridDim.x * PM_WARPS, pipe = blockIdx.x * PM_WARPS + w;
    const uint32_t mine = pipe < total ? (total - pipe + npipes - 1) / npipes : 0;
    auto issue_load = [&](uint32_t i) {
        const uint32_t u = pipe + i * npipes, m = u / a.units_per_page, c = u % a.units_per_page;
        const int s = (int)(i % PM_STAGES);
        const uint32_t bar = smem_u32(&bars[w][s]);
        mbar_expect_tx(bar, chunk);
        bulk_g2s(smem_u32(ring + (size_t)s * chunk), a.src[m] + ((size_t)c << a.log2c), chunk, bar);
    };
    const uint32_t pre = mine < PM_STAGES ? mine : PM_STAGES;
    for (uint32_t i = 0; i < pre; ++i) issue_load(i);
    for (uint32_t i = 0; i < mine; ++i) {
        const int s = (int)(i % PM_STAGES);
        mbar_wait(smem_u32(&bars[w][s]), (i / PM_STAGES) & 1);
        const uint32_t u = pipe + i * npipes, m = u / a.units_per_page, c = u % a.units_per_page;
        bulk_s2g(a.dst[m] + ((size_t)c << a.log2c), smem_u32(ring + (size_t)s * chunk), chunk);
        bulk_commit();
        if (i >= 1 && i - 1 + PM_STAGES < mine) {
            bulk_wait_read<1>();
            issue_load(i - 1 + PM_STAGES);
        }
    }
    bulk_wait_all();
}

// The switch: the blocks that live in VA page v are blockperm[v * bpp + k]; their table entries (and the page's offset) now
// point into the other half.  One CTA per move.
__global__ void page_switch_kernel(const __grid_constant__ PageMoveArgs a, const uint32_t* __restrict__ blockperm,
                                   uint32_t* __restrict__ T, uint32_t* __restrict__ pageoff, uint32_t bpp, uint32_t nb) {
    const uint32_t m = blockIdx.x;
    if (m >= a.n) return;
    const uint32_t v = a.v[m], off = a.newoff[m];
    for (uint32_t k = threadIdx.x; k < bpp; k += blockDim.x) {
        const uint32_t slot = v * bpp + k, i = blockperm[slot];
        if (i < nb) T[i] = slot + off;
    }
    if (threadIdx.x == 0) pageoff[v] = off;
}

static void give_back_event(RekeyPages* rk, cudaEvent_t e) { rk->events.push_back(e); }
static cloak_status take_event(RekeyPages* rk, cudaEvent_t* e) {
    if (!rk->events.empty()) {
        *e = rk->events.back();
        rk->events.pop_back();
        return CLOAK_OK;
    }
    CLOAK_CUDA(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    return CLOAK_OK;
}

// Moves whose switch has been passed by the stream: unmap the old address, the physical page is free.
static cloak_status retire(cloak_pool* p, bool wait) {
    RekeyPages* rk = p->rk;
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    size_t keep = 0;
    for (size_t i = 0; i < rk->inflight.size(); ++i) {
        PageMove& m = rk->inflight[i];
        cudaError_t q = wait ? cudaEventSynchronize(m.done) : cudaEventQuery(m.done);
        if (q == cudaErrorNotReady) {
            cudaGetLastError();
            rk->inflight[keep++] = m;
            continue;
        }
        if (q != cudaSuccess) return fail(CLOAK_ERR_CUDA, "rekey_pages: event: %s", cudaGetErrorString(q));
        CLOAK_CU(d->MemUnmap((CUdeviceptr)p->page_va(m.v, m.old_half), p->page));
        rk->free_pages.push_back(m.from);
        rk->moving[m.v] = 0;
        if (rk->cur[m.v] == rk->tgt[m.v]) --rk->todo;
        give_back_event(rk, m.done);
    }
    rk->inflight.resize(keep);
    return CLOAK_OK;
}

// Up to max_moves new moves: every free physical page of the pool takes the VA page that wants it; a free SPARE takes the
// next page that starts a new cycle.
static cloak_status issue(cloak_pool* p, uint32_t max_moves, cudaStream_t s) {
    RekeyPages* rk = p->rk;
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    CUmemAccessDesc acc = {};
    acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    acc.location.id = p->device;
    acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
    PageMoveArgs a;
    a.n = 0;
    a.log2c = 13;
    a.units_per_page = (uint32_t)(p->page >> a.log2c);
    std::vector<PageMove> batch;
    const uint32_t np = p->npages;
    if (max_moves > (uint32_t)PM_MAX) max_moves = PM_MAX;
    for (size_t f = 0; f < rk->free_pages.size() && batch.size() < max_moves;) {
        const uint32_t F = rk->free_pages[f];
        uint32_t v = 0xffffffffu;
        if (F < np) {
            const uint32_t u = rk->want[F];
            if (!rk->moving[u] && rk->cur[u] != F) v = u;      // (cur[u] == F cannot be: F is free)
        } else {
            // a spare: park the next page whose own target is still occupied (a page whose target is free is served above)
            for (uint32_t tries = 0; tries < np; ++tries) {
                const uint32_t c = rk->scan;
                rk->scan = rk->scan + 1 == np ? 0 : rk->scan + 1;
                if (rk->cur[c] != rk->tgt[c] && !rk->moving[c] && rk->cur[c] < np &&
                    std::find(rk->free_pages.begin(), rk->free_pages.end(), rk->tgt[c]) == rk->free_pages.end()) {
                    v = c;
                    break;
                }
            }
        }
        if (v == 0xffffffffu) { ++f; continue; }
        const uint32_t nh = p->page_half[v] ^ 1u;
        const CUdeviceptr dst = (CUdeviceptr)p->page_va(v, nh);
        CLOAK_CU(d->MemMap(dst, p->page, 0, p->handles[F], 0));
        CLOAK_CU(d->MemSetAccess(dst, p->page, &acc, 1));
        PageMove m;
        m.v = v;
        m.from = rk->cur[v];
        m.to = F;
        m.old_half = p->page_half[v];
        m.done = nullptr;
        a.src[a.n] = p->page_va(v, m.old_half);
        a.dst[a.n] = (char*)dst;
        a.v[a.n] = v;
        a.newoff[a.n] = nh * p->nslots;
        ++a.n;
        rk->cur[v] = F;
        rk->moving[v] = 1;
        p->page_half[v] = (uint8_t)nh;
        batch.push_back(m);
        rk->free_pages.erase(rk->free_pages.begin() + f);            // (f now indexes the next free page)
    }
    if (batch.empty()) return CLOAK_OK;
    static std::atomic<uint64_t> opted{0};
    const size_t smem = (size_t)PM_WARPS * PM_STAGES << a.log2c;
    if (cloak_status ost = smem_opt_in(page_copy_kernel, smem, p->device, opted)) return ost;
    const uint32_t units = a.n * a.units_per_page;
    uint32_t ctas = (units + PM_WARPS - 1) / PM_WARPS;
    const uint32_t sms = (uint32_t)sm_count(p->device);
    if (ctas > sms) ctas = sms;
    p->wrote(s);
    page_copy_kernel<<<ctas, PM_WARPS * 32, smem, s>>>(a);
    launched();
    page_switch_kernel<<<a.n, 128, 0, s>>>(a, p->d_blockperm, p->d_T, p->d_pageoff, p->bpp, p->nb);
    launched();
    CLOAK_LAUNCH_CHECK();
    cudaEvent_t ev;
    if (cloak_status est = take_event(rk, &ev)) return est;
    CLOAK_CUDA(cudaEventRecord(ev, s));
    // one event serves the whole batch: every move gets its own handle to it only through the first; the others share
    for (size_t i = 0; i < batch.size(); ++i) {
        if (i == 0) batch[i].done = ev;
        else {
            cudaEvent_t e2;
            if (cloak_status est = take_event(rk, &e2)) return est;
            CLOAK_CUDA(cudaEventRecord(e2, s));
            batch[i].done = e2;
        }
        rk->inflight.push_back(batch[i]);
    }
    rk->moves_issued += (uint32_t)batch.size();
    return CLOAK_OK;
}

// When every page is home: the spares are free again -- release them, publish the new page map.
static cloak_status finish(cloak_pool* p, cudaStream_t s) {
    RekeyPages* rk = p->rk;
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    for (uint32_t k = 0; k < rk->nspare; ++k) d->MemRelease(p->handles[p->npages + k]);
    p->handles.resize(p->npages);
    p->h_pageinv = rk->tgt;
    p->h_pageperm = rk->want;
    // the host vectors live in the pool: the copies below read them when the stream gets there (pageable source: the
    // runtime stages it before the call returns)
    CLOAK_CUDA(cudaMemcpyAsync(p->d_pageperm, p->h_pageperm.data(), (size_t)p->npages * 4, cudaMemcpyHostToDevice, s));
    CLOAK_CUDA(cudaMemcpyAsync(p->d_pageinv, p->h_pageinv.data(), (size_t)p->npages * 4, cudaMemcpyHostToDevice, s));
    if (p->alias) {                                       // the dump view's alias mapping is in creation order: still valid
    }
    for (cudaEvent_t e : rk->events) cudaEventDestroy(e);
    delete rk;
    p->rk = nullptr;
    return CLOAK_OK;
}

void rekey_pages_abandon(cloak_pool* p) {
    RekeyPages* rk = p->rk;
    if (!rk) return;
    const DriverApi* d = driver();
    cudaDeviceSynchronize();
    if (d) {
        for (PageMove& m : rk->inflight) d->MemUnmap((CUdeviceptr)p->page_va(m.v, m.old_half), p->page);
        // (the pages' current addresses are unmapped by the pool's own teardown, spares included in p->handles)
    }
    for (PageMove& m : rk->inflight) cudaEventDestroy(m.done);
    for (cudaEvent_t e : rk->events) cudaEventDestroy(e);
    delete rk;
    p->rk = nullptr;
}

}  // namespace cloak

using namespace cloak;

extern "C" cloak_status cloak_rekey_pages_begin(cloak_pool* pool, uint64_t new_key, uint32_t spare_pages, void* stream) {
    if (!pool) return fail(CLOAK_ERR_INVALID, "rekey_pages_begin: NULL pool");
    if (!pool->vmm) return fail(CLOAK_ERR_UNSUPPORTED, "rekey_pages_begin: the pool has no real (VMM) pages");
    if (pool->flags & CLOAK_POOL_IDENTITY) return fail(CLOAK_ERR_INVALID, "rekey_pages_begin: an identity pool has no key");
    if (pool->rk) return fail(CLOAK_ERR_INVALID, "rekey_pages_begin: a page re-key of this pool is already in progress");
    if (spare_pages == 0) spare_pages = 1;
    if (spare_pages > 64) return fail(CLOAK_ERR_INVALID, "rekey_pages_begin: at most 64 spare pages");
    DeviceGuard g(pool->device);
    const DriverApi* d = driver();
    if (!d) return CLOAK_ERR_CUDA;
    cudaStream_t s = (cudaStream_t)stream;
    const uint32_t np = pool->npages;
    // the new page map: the same keygen as cloak_pool_create, on the device, read back (npages entries)
    AsyncBuf tab(s);
    if (cloak_status ast = tab.alloc((size_t)2 * np * 4)) return ast;
    uint32_t* d_new = static_cast<uint32_t*>(tab.p);
    if (cloak_status st = keygen_device(new_key, 2ull << 32, np, d_new, d_new + np, s)) return st;
    RekeyPages* rk = new (std::nothrow) RekeyPages();
    if (!rk) return fail(CLOAK_ERR_OOM, "rekey_pages_begin: host allocation failed");
    rk->want.resize(np);
    rk->tgt.resize(np);
    cudaError_t e = cudaMemcpyAsync(rk->want.data(), d_new, (size_t)np * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(rk->tgt.data(), d_new + np, (size_t)np * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {
        delete rk;
        return fail(CLOAK_ERR_CUDA, "rekey_pages_begin: %s", cudaGetErrorString(e));
    }
    CUmemAllocationProp prop = {};
    prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
    prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    prop.location.id = pool->device;
    for (uint32_t k = 0; k < spare_pages; ++k) {
        CUmemGenericAllocationHandle h;
        CUresult r = d->MemCreate(&h, pool->page, &prop, 0);
        if (r != CUDA_SUCCESS) {
            for (uint32_t j = 0; j < k; ++j) d->MemRelease(pool->handles[np + j]);
            pool->handles.resize(np);
            delete rk;
            return fail(r == CUDA_ERROR_OUT_OF_MEMORY ? CLOAK_ERR_OOM : CLOAK_ERR_CUDA, "rekey_pages_begin: cuMemCreate: %s", cu_err(r));
        }
        pool->handles.push_back(h);
        rk->free_pages.push_back(np + k);
    }
    rk->new_key = new_key;
    rk->nspare = spare_pages;
    rk->cur = pool->h_pageinv;
    rk->moving.assign(np, 0);
    for (uint32_t v = 0; v < np; ++v)
        if (rk->cur[v] != rk->tgt[v]) ++rk->todo;
    pool->rk = rk;
    pool->key = new_key;          // (the BLOCK tables keep the key they were drawn with; pool->key names the page map's from here on)
    return CLOAK_OK;
}

extern "C" cloak_status cloak_rekey_pages_step(cloak_pool* pool, uint32_t max_moves, void* stream, uint32_t* h_remaining) {
    if (!pool) return fail(CLOAK_ERR_INVALID, "rekey_pages_step: NULL pool");
    if (!pool->rk) {
        if (h_remaining) *h_remaining = 0;
        return CLOAK_OK;
    }
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    if (cloak_status st = retire(pool, false)) return st;
    if (pool->rk->todo > 0 && max_moves > 0)
        if (cloak_status st = issue(pool, max_moves, s)) return st;
    const uint32_t left = pool->rk->todo;
    if (left == 0 && pool->rk->inflight.empty()) {
        if (cloak_status st = finish(pool, s)) return st;
    }
    if (h_remaining) *h_remaining = left + (pool->rk ? (uint32_t)pool->rk->inflight.size() : 0);
    return CLOAK_OK;
}

extern "C" cloak_status cloak_rekey_pages_finish(cloak_pool* pool, void* stream) {
    if (!pool) return fail(CLOAK_ERR_INVALID, "rekey_pages_finish: NULL pool");
    DeviceGuard g(pool->device);
    cudaStream_t s = (cudaStream_t)stream;
    while (pool->rk) {
        if (cloak_status st = retire(pool, true)) return st;            // waits for the moves in flight
        if (pool->rk->todo > 0) {
            if (cloak_status st = issue(pool, PM_MAX, s)) return st;
        } else if (pool->rk->inflight.empty()) {
            if (cloak_status st = finish(pool, s)) return st;
        }
    }
    CLOAK_CUDA(cudaStreamSynchronize(s));
    return CLOAK_OK;
}
