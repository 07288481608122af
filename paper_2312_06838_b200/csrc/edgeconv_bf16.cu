// edgeconv_bf16.cu -- placeholder until the tcgen05 path lands (next commit): GNN_BF16 models are refused.
#include "gnn_internal.h"
int edgeconv_bf16_prepare(gnn_model&, const float*) { return GNN_ERR_BAD_ARCH; }
int launch_edgeconv_bf16(gnn_model&, int, const float*, const int32_t*, int, float*, Workspace&, cudaStream_t) { return GNN_ERR_BAD_ARCH; }
