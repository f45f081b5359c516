// S7 cloak_gemm: placeholder until the tcgen05 kernel lands (returns CLOAK_ERR_UNSUPPORTED).
#include "common.cuh"
extern "C" cloak_status cloak_gemm(const cloak_pool* pool, const cloak_tensor* w, const void* d_x, void* d_y,
                                   uint32_t batch, void* stream) {
    (void)pool; (void)w; (void)d_x; (void)d_y; (void)batch; (void)stream;
    return cloak::fail(CLOAK_ERR_UNSUPPORTED, "gemm: not implemented yet");
}
