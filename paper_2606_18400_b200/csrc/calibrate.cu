// Per-SM streaming weights: how fast each SM of THIS device pulls a read stream out of HBM.
//
// Why.  The decode GEMV is a read stream that should end on all SMs at once (the reader is bandwidth-
// bound).  On B200 the SMs do not stream equally fast: with the same bytes in flight per SM (192 KiB of bulk copies), a
// dynamic chunk queue hands some SMs 1.7 x the work of others -- 348 .. 608 of 65 536 chunks, in three tiers (SM pairs of a
// TPC always agree), reproducible from run to run (correlation 0.97) and following the physical position of the SM (which
// GPC / how many neighbours share its path to L2), i.e. a property of the individual part.  Equal static shares therefore
// finish when the slowest tier does: 3 % later than the queue on a 2 GiB stream, and at every grid-wide dependency of a
// chain the fast SMs wait for the slow ones.  Measured once per device, the weights let a kernel cut its work into STATIC
// shares proportional to speed: balanced like the queue, with no atomics on the producer's path and a split that is
// fixed for the life of the process (deterministic results).
//
// Result (round 2, B200): the weights are real and stable, but the streaming GEMV does NOT profit from
// them: its SMs are not limited by the contended path to L2 but by their own ring (bytes in flight / loaded latency, the
// stage also being held while the consumers work through it), so with equal shares all 148 producers already end within
// 4 us of each other (68 .. 72 us of a 75 us launch), and weighted shares make the "fast" SMs finish LAST: cfg1 layer
// 79.9 -> 85.5 us (batch 1), 93.7 -> 101.9 us (batch 16).  A pure read stream of large pieces, which does saturate the path,
// gains 6 % from a dynamic queue over equal shares (58.9 vs 62.4 us for 436 MB).  The weighted split was then taken OUT of the
// GEMV kernel again: merely carrying the switch (a flag test, a table load and 64-bit range arithmetic per op in producer and
// consumers) cost cfg2's decode chain 2 % and a 12-layer MoE chain of 348 small ops 12 % (0.462 -> 0.526 ms).  What stays is the
// measurement itself, as a report: cloak_sm_weights.
//
// How.  One CTA per SM (192 KiB of shared memory each) draws 32 KiB chunks of a scratch buffer from an atomic counter and
// pulls them with cp.async.bulk through a 6-stage ring; chunks drawn per %smid over two measured passes = the weight.
// Quantised to 1/64 of the mean so that run-to-run noise (~1 %) rarely moves a share.  The table handed to kernels is
// cum[0 .. nsm] in 16-bit fixed point (cum[nsm] = 65536), indexed by %smid: SM s owns units [n*cum[s] >> 16, n*cum[s+1] >> 16).
#include <mutex>
#include "common.cuh"
#include "async.cuh"

namespace cloak {

constexpr int CAL_STAGES = 6;
constexpr uint32_t CAL_CHUNK = 32768;

__global__ void __launch_bounds__(32, 1) sm_stream_rate_kernel(const char* src, uint32_t chunks_in_buf, uint32_t nchunks,
                                                               uint32_t* counter, uint32_t* per_smid, uint32_t* seen) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full[CAL_STAGES];
    if (threadIdx.x != 0) return;
    for (int s = 0; s < CAL_STAGES; ++s) mbar_init(smem_u32(&full[s]), 1);
    fence_barrier_init();
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    const uint32_t base = smem_u32(smem);
    auto issue = [&](int s, uint32_t c) {
        mbar_expect_tx(smem_u32(&full[s]), CAL_CHUNK);
        bulk_g2s(base + s * CAL_CHUNK, src + (size_t)(c % chunks_in_buf) * CAL_CHUNK, CAL_CHUNK, smem_u32(&full[s]));
    };
    uint32_t issued = 0, done = 0;
    for (int s = 0; s < CAL_STAGES; ++s) {
        const uint32_t c = atomicAdd(counter, 1u);
        if (c >= nchunks) break;
        issue(s, c);
        ++issued;
    }
    bool more = issued == CAL_STAGES;
    uint32_t s = 0, ph = 0;
    while (done < issued) {
        mbar_wait(smem_u32(&full[s]), ph);
        ++done;
        if (more) {
            const uint32_t c = atomicAdd(counter, 1u);
            if (c < nchunks) { issue((int)s, c); ++issued; } else more = false;
        }
        if (++s == CAL_STAGES) { s = 0; ph ^= 1; }
    }
    atomicAdd(per_smid + smid, done);
    atomicAdd(seen + smid, 1u);
}

struct SmWeights {
    std::atomic<int> state{0};      // 0 not measured, 1 ready, -1 unusable (measurement failed or SM ids are not 0 .. nsm-1, one CTA each)
    uint32_t nsm = 0;
    uint32_t* d_cum = nullptr;      // device, nsm + 1 entries
    std::vector<float> w;           // relative speed, mean 1
};
static SmWeights g_smw[64];
static std::mutex g_smw_mu;

static void measure(int device, SmWeights& out) {
    out.state.store(-1);
    const int nsm = sm_count(device);
    if (nsm <= 1 || nsm > 1024) return;
    const size_t buf_bytes = 1ull << 30;
    const uint32_t in_buf = (uint32_t)(buf_bytes / CAL_CHUNK), nchunks = 2 * in_buf;      // 2 GiB per pass
    char* buf = nullptr;
    uint32_t* d = nullptr;                                                                 // counter | per_smid[1024] | seen[1024]
    if (cudaMalloc((void**)&buf, buf_bytes) != cudaSuccess) { cudaGetLastError(); return; }
    if (cudaMalloc((void**)&d, (1 + 2048) * 4) != cudaSuccess) { cudaGetLastError(); cudaFree(buf); return; }
    const size_t smem = (size_t)CAL_STAGES * CAL_CHUNK;
    bool ok = cudaFuncSetAttribute(sm_stream_rate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess;
    std::vector<uint32_t> h(1 + 2048, 0);
    for (int pass = 0; pass < 3 && ok; ++pass) {
        // pass 0 warms up (and its counts are thrown away with this memset); passes 1 and 2 accumulate
        if (pass <= 1) ok = cudaMemset(d, 0, (1 + 2048) * 4) == cudaSuccess;
        else ok = cudaMemset(d, 0, 4) == cudaSuccess;
        if (!ok) break;
        sm_stream_rate_kernel<<<nsm, 32, smem>>>(buf, in_buf, nchunks, d, d + 1, d + 1 + 1024);
        launched();
        ok = cudaDeviceSynchronize() == cudaSuccess;
    }
    ok = ok && cudaMemcpy(h.data(), d, h.size() * 4, cudaMemcpyDeviceToHost) == cudaSuccess;
    cudaFree(buf);
    cudaFree(d);
    if (!ok) { cudaGetLastError(); return; }
    // every SM id 0 .. nsm-1 exactly once per pass, nothing outside: the kernels may then index the table by %smid
    double total = 0;
    for (int s = 0; s < 1024; ++s) {
        const uint32_t cnt = h[1 + s], seen = h[1 + 1024 + s];
        if (s < nsm ? (seen != 2 || cnt == 0) : (seen != 0)) return;
        if (s < nsm) total += cnt;
    }
    const double mean = total / nsm;
    out.w.resize(nsm);
    std::vector<uint32_t> cum(nsm + 1, 0);
    double qsum = 0;
    for (int s = 0; s < nsm; ++s) {
        double q = (double)(long)(h[1 + s] / mean * 64.0 + 0.5) / 64.0;       // quantised to 1/64 of the mean
        if (q < 0.25) q = 0.25;
        out.w[s] = (float)q;
        qsum += q;
    }
    double run = 0;
    for (int s = 0; s < nsm; ++s) {
        cum[s] = (uint32_t)(run / qsum * 65536.0 + 0.5);
        run += out.w[s];
    }
    cum[nsm] = 65536;
    for (int s = 0; s < nsm; ++s) out.w[s] = (float)(out.w[s] * nsm / qsum);
    if (cudaMalloc((void**)&out.d_cum, (nsm + 1) * 4) != cudaSuccess ||
        cudaMemcpy(out.d_cum, cum.data(), (nsm + 1) * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return;
    }
    out.nsm = (uint32_t)nsm;
    out.state.store(1, std::memory_order_release);
}

// Measured at most once per device and process; call with the device current, outside stream capture.
static void ensure_sm_weights(int device) {
    if (device < 0 || device >= 64) return;
    std::lock_guard<std::mutex> lock(g_smw_mu);
    if (g_smw[device].state.load() == 0) measure(device, g_smw[device]);
}

}  // namespace cloak

extern "C" cloak_status cloak_sm_weights(int device, uint32_t capacity, float* h_weights, uint32_t* h_nsm) {
    using namespace cloak;
    if (device < 0 || device >= 64 || !h_nsm) return fail(CLOAK_ERR_INVALID, "sm_weights: bad device or NULL h_nsm");
    {
        DeviceGuard g(device);
        if (!g.ok) return fail(CLOAK_ERR_CUDA, "sm_weights: cannot select device %d", device);
        ensure_sm_weights(device);
    }
    const SmWeights& w = g_smw[device];
    if (w.state.load() != 1) {
        *h_nsm = 0;
        return CLOAK_OK;                       // not usable on this device: kernels use equal shares
    }
    *h_nsm = w.nsm;
    if (h_weights) {
        if (capacity < w.nsm) return fail(CLOAK_ERR_INVALID, "sm_weights: room for %u weights, the device has %u SMs", capacity, w.nsm);
        for (uint32_t s = 0; s < w.nsm; ++s) h_weights[s] = w.w[s];
    }
    return CLOAK_OK;
}
