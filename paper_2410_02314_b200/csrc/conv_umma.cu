#include <cstdio>
#include "smlm_internal.cuh"
namespace smlm {
struct UmmaPlan { int dummy; };
size_t umma_packed_weight_bytes(int C) { return 16; }
void umma_pack_weights_host(int, const float*, void*) {}
UmmaPlan* umma_plan_create(const void*, const void*, ActShape, int, char* err, size_t n) { snprintf(err, n, "stub"); return nullptr; }
void umma_plan_destroy(UmmaPlan*) {}
cudaError_t launch_conv_umma(UmmaPlan*, int, int, const void*, const float*, int, cudaStream_t, char*, size_t) { return cudaErrorNotSupported; }
}
