// tina_umma.cu -- tcgen05 tensor-core path (placeholder until the fused kernel lands).
#include "tina_common.cuh"
namespace tina {
bool umma_supported(int, bool) { return false; }
tina_status umma_pfb(const void*, int, long long, int, int, const float*, bool, bool, tina_precision,
                     void*, cudaStream_t) { return fail(TINA_ERR_UNSUPPORTED, "tensor path not built"); }
void umma_clear_plans() {}
}
