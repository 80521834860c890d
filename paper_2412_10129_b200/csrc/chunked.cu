// chunked.cu — single-GPU host-chunking path (§2.5). Placeholder:
// the streaming implementation lands after the in-HBM kernels are parity-green.
#include "common.cuh"
namespace tg {
static size_t g_budget = 0;
size_t chunk_budget() { return g_budget; }
int chunked_ax(const float*, const tigre_geo*, const double*, int, int, float*, cudaStream_t) { return TIGRE_ERR_MEMSPACE; }
int chunked_atb(const float*, const tigre_geo*, const double*, int, int, float*, cudaStream_t) { return TIGRE_ERR_MEMSPACE; }
}  // namespace tg
extern "C" int tigre_set_chunk_budget(size_t bytes) { tg::g_budget = bytes; return TIGRE_OK; }
