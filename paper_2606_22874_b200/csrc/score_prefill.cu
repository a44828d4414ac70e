#include "common.cuh"
namespace spot {
spot_status score_prefill(const spot_select_params*, float*, int, cudaStream_t) { return SPOT_ERR_UNSUPPORTED; }
}
