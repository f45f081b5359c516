// Error plumbing, driver-API loader, host-side tensor-order planner (S3).
#include <stdarg.h>
#include <string.h>
#include <algorithm>
#include <mutex>
#include "common.cuh"

namespace cloak {

static thread_local char g_err[512] = "";
std::atomic<unsigned long long> g_launches{0};

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

cloak_status fail(cloak_status st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

static DriverApi g_drv;
static bool g_drv_ok = false;
static std::once_flag g_drv_once;

template <typename F>
static bool load_sym(F& fn, const char* name) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q);
    if (e != cudaSuccess || p == nullptr || q != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    fn = reinterpret_cast<F>(p);
    return true;
}

const DriverApi* driver() {
    std::call_once(g_drv_once, [] {
        bool ok = true;
        ok &= load_sym(g_drv.MemGetAllocationGranularity, "cuMemGetAllocationGranularity");
        ok &= load_sym(g_drv.MemAddressReserve, "cuMemAddressReserve");
        ok &= load_sym(g_drv.MemAddressFree, "cuMemAddressFree");
        ok &= load_sym(g_drv.MemCreate, "cuMemCreate");
        ok &= load_sym(g_drv.MemRelease, "cuMemRelease");
        ok &= load_sym(g_drv.MemMap, "cuMemMap");
        ok &= load_sym(g_drv.MemUnmap, "cuMemUnmap");
        ok &= load_sym(g_drv.MemSetAccess, "cuMemSetAccess");
        ok &= load_sym(g_drv.GetErrorString, "cuGetErrorString");
        ok &= load_sym(g_drv.TensorMapEncodeTiled, "cuTensorMapEncodeTiled");
        g_drv_ok = ok;
    });
    if (!g_drv_ok) {
        set_error("CUDA driver API unavailable (no driver / no device)");
        return nullptr;
    }
    return &g_drv;
}

const char* cu_err(CUresult r) {
    const char* s = nullptr;
    if (g_drv_ok && g_drv.GetErrorString(r, &s) == CUDA_SUCCESS && s) return s;
    return "CUDA driver error";
}

int sm_count(int device) {
    static int cached[64] = {0};
    if (device < 0 || device >= 64) return 148;
    if (cached[device] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || n <= 0) {
            cudaGetLastError();
            n = 148;
        }
        cached[device] = n;
    }
    return cached[device];
}

// ---- the library's stream-ordered memory pool, one per device
static cudaMemPool_t g_mempool[64];
static std::mutex g_mempool_mu;

cloak_status async_alloc(void** p, size_t bytes, cudaStream_t s) {
    int dev = 0;
    CLOAK_CUDA(cudaGetDevice(&dev));
    cudaMemPool_t mp = nullptr;
    if (dev >= 0 && dev < 64) {
        std::lock_guard<std::mutex> lock(g_mempool_mu);
        if (!g_mempool[dev]) {
            cudaMemPoolProps props = {};
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = dev;
            cudaMemPool_t np = nullptr;
            if (cudaMemPoolCreate(&np, &props) == cudaSuccess) {
                uint64_t keep = 512ull << 20;      // freed scratch stays cached up to this much; the rest goes back at a sync
                cudaMemPoolSetAttribute(np, cudaMemPoolAttrReleaseThreshold, &keep);
                g_mempool[dev] = np;
            }
            cudaGetLastError();
        }
        mp = g_mempool[dev];
    }
    if (mp) CLOAK_CUDA(cudaMallocFromPoolAsync(p, bytes, mp, s));
    else CLOAK_CUDA(cudaMallocAsync(p, bytes, s));
    return CLOAK_OK;
}

// ---- host Philox4x32-10 for the tiny tensor-order permutation of S3.
static inline void philox_host(uint32_t c[4], uint32_t k0, uint32_t k1) {
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = 0xD2511F53ull * c[0], p1 = 0xCD9E8D57ull * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1, n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
}

void keygen_host(uint64_t key, uint64_t stream_id, uint32_t n, std::vector<uint32_t>& perm) {
    std::vector<uint64_t> r(n);
    for (uint32_t i = 0; i < n; ++i) {
        uint32_t c[4] = {i, 0u, (uint32_t)stream_id, (uint32_t)(stream_id >> 32)};
        philox_host(c, (uint32_t)key, (uint32_t)(key >> 32));
        r[i] = ((uint64_t)c[0] << 32) | c[1];
    }
    perm.resize(n);
    for (uint32_t i = 0; i < n; ++i) perm[i] = i;
    std::sort(perm.begin(), perm.end(), [&](uint32_t a, uint32_t b) {
        return r[a] != r[b] ? r[a] < r[b] : a < b;
    });
}

}  // namespace cloak

extern "C" const char* cloak_last_error(void) { return cloak::g_err; }

extern "C" uint64_t cloak_launch_count(void) { return cloak::g_launches.load(); }

extern "C" const char* cloak_version(void) { return "cloak-b200 0.2 sm_100a"; }

namespace cloak { int gemv_coop_pdl_state(); }
extern "C" const char* cloak_runtime_info(void) {
    static thread_local char buf[256];
    const int st = cloak::gemv_coop_pdl_state();
    snprintf(buf, sizeof(buf), "gemv_chain: cooperative launch where a chain has `after` ops (programmatic dependent launch %s), "
                               "plain launch + programmatic dependent launch elsewhere; kernels launched %llu",
             st < 0 ? "not probed yet" : (st ? "accepted with it" : "rejected with it (dropped)"),
             (unsigned long long)cloak::g_launches.load());
    return buf;
}

extern "C" cloak_status cloak_arena_plan(uint64_t key, uint32_t T, const uint64_t* h_bytes, uint32_t block_bytes,
                                         uint64_t* h_offsets_out, uint64_t* h_total_out) {
    if (T == 0 || !h_bytes || !h_offsets_out) return cloak::fail(CLOAK_ERR_INVALID, "arena_plan: null argument or T == 0");
    if (block_bytes < 16 || (block_bytes & 15)) return cloak::fail(CLOAK_ERR_ALIGN, "arena_plan: block_bytes must be a multiple of 16");
    std::vector<uint32_t> order;
    cloak::keygen_host(key, 3ull << 32, T, order);
    uint64_t at = 0;
    for (uint32_t p = 0; p < T; ++p) {
        uint32_t t = order[p];
        h_offsets_out[t] = at;
        at += (h_bytes[t] + block_bytes - 1) / block_bytes * (uint64_t)block_bytes;
    }
    if (h_total_out) *h_total_out = at;
    return CLOAK_OK;
}
