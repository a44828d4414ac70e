#include "common.cuh"
extern "C" size_t spot_sparse_attn_prefill_workspace_bytes(const spot_attn_params*) { return 0; }
extern "C" spot_status spot_sparse_attn_prefill(const spot_attn_params*, void*) { return SPOT_ERR_UNSUPPORTED; }
