// tcgen05 / TMEM tensor-core MLP kernels (bf16 and int8).  Placeholder until the first version lands.
#include "etx_internal.h"
namespace etx {
bool umma_supported(const etx_ctx*) { return false; }
void umma_configure(etx_ctx*) {}
void launch_embed_umma(etx_ctx*, int, cudaStream_t) {}
void launch_gnn_mlp_umma(etx_ctx*, int, int, int, bool, cudaStream_t) {}
}  // namespace etx
