// Step a3' -- block-sparse causal GQA flash attention for chunked prefill (Fig. 2):
// every 64-token query block attends to its own list of selected 64-token key blocks; only the diagonal block needs a
// token-level mask (t <= own position).  This file holds the C-ABI entry and its host-side argument checks; the
// kernel (tcgen05 / TMEM / TMA) is in attn_prefill_tc.cu.  (Round 1's first form of this step was an mma.sync flash
// kernel at 328 TFLOP/s; profiles/r1_prefill_cfg5.md keeps its numbers.)
#include "common.cuh"

namespace spot {

namespace {

spot_status check_prefill(const spot_attn_params* p) {
    if (!p || !p->q || !p->k || !p->v || !p->out) return SPOT_ERR_INVALID_ARG;
    if (!aligned16(p->q) || !aligned16(p->k) || !aligned16(p->v) || !aligned16(p->out)) return SPOT_ERR_INVALID_ARG;
    if (p->B <= 0 || p->H_q <= 0 || p->H_kv <= 0 || p->H_q % p->H_kv != 0) return SPOT_ERR_INVALID_ARG;
    if (p->Tq <= 0 || p->Tq % 64 != 0 || p->q_start < 0 || p->q_start % 64 != 0) return SPOT_ERR_INVALID_ARG;   // R26
    if (p->H_q / p->H_kv > 16) return SPOT_ERR_UNSUPPORTED;
    if (p->D != 128 || (p->blk != 64 && p->blk != 16)) return SPOT_ERR_UNSUPPORTED;
    if (p->page_table) {          // f3 / R32: a 64-token block must sit inside one page
        if (p->page_tokens <= 0 || p->page_tokens % 16 != 0 || p->kv_stride_batch <= 0) return SPOT_ERR_INVALID_ARG;
        if (p->page_tokens % 64 != 0) return SPOT_ERR_UNSUPPORTED;
        if ((int64_t)p->page_table_stride * p->page_tokens < (int64_t)p->q_start + p->Tq) return SPOT_ERR_INVALID_ARG;
    }
    if (p->kv_stride_token < p->D || p->kv_stride_token % 8 || p->kv_stride_head % 8 || p->kv_stride_batch % 8)
        return SPOT_ERR_INVALID_ARG;
    if (p->indices && (!p->budgets || p->cap <= 0)) return SPOT_ERR_INVALID_ARG;
    return SPOT_OK;
}

}  // namespace

}  // namespace spot

namespace spot { spot_status attn_prefill_tc(const spot_attn_params* p, cudaStream_t stream); }

using namespace spot;

extern "C" size_t spot_sparse_attn_prefill_workspace_bytes(const spot_attn_params* p) {
    (void)p;
    return 0;   // the prefill form keeps all of its state on chip
}

extern "C" spot_status spot_sparse_attn_prefill(const spot_attn_params* p, void* stream) {
    spot_status st = check_prefill(p);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    return attn_prefill_tc(p, (cudaStream_t)stream);
}
