// C-ABI glue: status strings, device check, spot_select orchestration (score kernel -> selection kernel) and the
// host-buffer decode step.  All argument validation happens here, on the host, before any launch.
#include "common.cuh"

namespace spot {

static thread_local int g_last_cuda_error = 0;
void set_last_cuda_error(int e) { g_last_cuda_error = e; }

spot_status check_device() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_last_cuda_error((int)e); return SPOT_ERR_CUDA; }
    static thread_local int cached_dev = -1, cached_major = 0;
    if (cached_dev != dev) {
        int major = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) { set_last_cuda_error((int)e); return SPOT_ERR_CUDA; }
        cached_dev = dev; cached_major = major;
    }
    return cached_major == 10 ? SPOT_OK : SPOT_ERR_UNSUPPORTED;
}

int sm_count() {
    static thread_local int cached = 0;
    if (!cached) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) cached = n;
        else cached = 148;
    }
    return cached;
}

// kernels implemented in the other translation units
spot_status score_decode(const spot_select_params* p, float* scores, int nb_stride, cudaStream_t s);
spot_status score_prefill(const spot_select_params* p, float* scores, int nb_stride, cudaStream_t s);
spot_status run_select(const spot_select_params* p, const float* scores, int nb_stride, int rows_per_seq, int max_nb,
                       cudaStream_t s);
spot_status check_attn_decode_args(const spot_attn_params* p);     // attn_decode.cu: the host-side checks of a3

namespace {

struct SelectGeom {
    int rows_per_seq;
    int max_nb;       // largest number of visible blocks of any row
    int nb_stride;    // row stride of the score matrix actually used
    bool own_scores;  // scores live in the workspace
};

spot_status select_geometry(const spot_select_params* p, SelectGeom* g, bool score_only = false) {
    if (!p) return SPOT_ERR_INVALID_ARG;
    if (!p->sel_q || !p->w || !p->sel_k) return SPOT_ERR_INVALID_ARG;
    if (score_only ? !p->block_scores : (!p->indices || !p->budgets)) return SPOT_ERR_INVALID_ARG;
    if (!aligned16(p->sel_q) || !aligned16(p->sel_k) || !aligned16(p->w)) return SPOT_ERR_INVALID_ARG;
    if (p->fmt != SPOT_SELK_BF16 && p->fmt != SPOT_SELK_INT4_E4M3 && p->fmt != SPOT_SELK_MXFP4 &&
        p->fmt != SPOT_SELK_FP8_E4M3) return SPOT_ERR_INVALID_ARG;
    if (p->mode != SPOT_MODE_TOPK && p->mode != SPOT_MODE_DUAL_TOPP) return SPOT_ERR_INVALID_ARG;
    if (p->B <= 0 || p->Tq <= 0 || p->H_idx <= 0 || p->d_idx <= 0 || p->d_idx % 32 != 0) return SPOT_ERR_INVALID_ARG;
    if (p->blk <= 0 || (!score_only && p->cap <= 0) || p->cache_stride_tokens <= 0) return SPOT_ERR_INVALID_ARG;
    if (p->sink_blocks < 0 || p->recency_blocks < 0 || p->kmin_blocks < 0 || p->top_k < 0) return SPOT_ERR_INVALID_ARG;
    if (p->mode == SPOT_MODE_DUAL_TOPP && !(p->p > 0.0 && p->p <= 1.0)) return SPOT_ERR_INVALID_ARG;
    if (!(p->temperature > 0.0)) return SPOT_ERR_INVALID_ARG;
    if (p->mode == SPOT_MODE_TOPK && p->top_k < p->sink_blocks + p->recency_blocks) return SPOT_ERR_INVALID_ARG;
    if (p->fmt != SPOT_SELK_BF16 && p->cache_stride_tokens % SELK_TILE != 0)
        return SPOT_ERR_INVALID_ARG;
    // 64-token blocks everywhere; the paper's own 16-token blocks (f3) at decode only
    if (p->blk != 64 && !(p->blk == 16 && p->q_block == 1)) return SPOT_ERR_UNSUPPORTED;
    int64_t max_tokens;
    if (p->q_block == 1) {
        if (p->Tq != 1 || !p->seq_len || p->max_seq_len <= 0) return SPOT_ERR_INVALID_ARG;
        if (p->max_seq_len > p->cache_stride_tokens) return SPOT_ERR_INVALID_ARG;
        g->rows_per_seq = 1;
        max_tokens = p->max_seq_len;
    } else if (p->q_block == 64) {
        if (p->Tq % 64 != 0 || p->q_start < 0 || p->q_start % 64 != 0) return SPOT_ERR_INVALID_ARG;
        if ((int64_t)p->q_start + p->Tq > p->cache_stride_tokens) return SPOT_ERR_INVALID_ARG;
        g->rows_per_seq = p->Tq / 64;
        max_tokens = (int64_t)p->q_start + p->Tq;
    } else {
        return SPOT_ERR_INVALID_ARG;
    }
    g->max_nb = (int)ceil_div64(max_tokens, p->blk);
    int need_cap = p->mode == SPOT_MODE_DUAL_TOPP ? g->max_nb : (p->top_k < g->max_nb ? p->top_k : g->max_nb);
    if (!score_only && p->cap < need_cap) return SPOT_ERR_INVALID_ARG;
    if (p->block_scores || p->block_probs) {
        if (p->nb_stride < g->max_nb) return SPOT_ERR_INVALID_ARG;
    }
    g->own_scores = p->block_scores == nullptr;
    g->nb_stride = g->own_scores ? ((g->max_nb + 3) & ~3) : p->nb_stride;
    return SPOT_OK;
}

// Prefill scoring of a quantised cache (f2): the visible prefix is dequantised into a BF16 scratch in the workspace and
// the BF16 tile-score GEMM runs on that (every dequantised value is exactly a BF16 number).  What the paper's own
// kernels do ("dequantisation overhead"); a fused unpack inside the GEMM's operand path is the next form.
size_t prefill_scratch_bytes(const spot_select_params* p) {
    if (p->q_block == 1 || p->fmt == SPOT_SELK_BF16) return 0;
    return 256 + (size_t)p->B * ((size_t)p->q_start + p->Tq) * p->H_idx * p->d_idx * 2;
}

spot_status score_any(const spot_select_params* p, float* scores, int nb_stride, void* scratch_area, cudaStream_t s) {
    if (p->q_block == 1) return score_decode(p, scores, nb_stride, s);
    if (p->fmt == SPOT_SELK_BF16) return score_prefill(p, scores, nb_stride, s);
    uint16_t* deq = reinterpret_cast<uint16_t*>((reinterpret_cast<uintptr_t>(scratch_area) + 255) & ~(uintptr_t)255);
    const int tok = p->q_start + p->Tq;
    spot_status st = spot_dequantize_selector_k(p->sel_k, deq, (spot_selk_format)p->fmt, p->B, tok, 0, p->cache_stride_tokens, p->H_idx,
                                                p->d_idx, (void*)s);
    if (st != SPOT_OK) return st;
    spot_select_params q = *p;
    q.sel_k = deq; q.fmt = SPOT_SELK_BF16; q.cache_stride_tokens = tok;
    return score_prefill(&q, scores, nb_stride, s);
}

}  // namespace

}  // namespace spot

using namespace spot;

extern "C" const char* spot_status_string(spot_status s) {
    switch (s) {
        case SPOT_OK: return "SPOT_OK";
        case SPOT_ERR_INVALID_ARG: return "SPOT_ERR_INVALID_ARG";
        case SPOT_ERR_UNSUPPORTED: return "SPOT_ERR_UNSUPPORTED";
        case SPOT_ERR_WORKSPACE_TOO_SMALL: return "SPOT_ERR_WORKSPACE_TOO_SMALL";
        case SPOT_ERR_CUDA: return "SPOT_ERR_CUDA";
    }
    return "SPOT_ERR_UNKNOWN";
}

extern "C" int spot_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" const char* spot_version(void) { return "0.2"; }
extern "C" size_t spot_struct_size(int which) {
    switch (which) {
        case 0: return sizeof(spot_select_params);
        case 1: return sizeof(spot_attn_params);
        case 2: return sizeof(spot_decode_step_host_params);
        case 3: return sizeof(spot_project_params);
    }
    return 0;
}

extern "C" size_t spot_select_workspace_bytes(const spot_select_params* p) {
    SelectGeom g;
    // a block without an index list is a spot_score_blocks block (it ignores indices / budgets / cap): size it as such
    if (!p || select_geometry(p, &g, /*score_only=*/!p->indices) != SPOT_OK) return 0;
    size_t bytes = 256;
    if (g.own_scores) bytes += (size_t)p->B * g.rows_per_seq * g.nb_stride * sizeof(float);
    return bytes + prefill_scratch_bytes(p);
}

extern "C" spot_status spot_select(const spot_select_params* p, void* stream) {
    SelectGeom g;
    spot_status st = select_geometry(p, &g);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    float* scores = p->block_scores;
    const size_t own = g.own_scores ? 256 + (size_t)p->B * g.rows_per_seq * g.nb_stride * sizeof(float) : 0;
    const size_t need = own + prefill_scratch_bytes(p);
    if (need && (!p->workspace || p->workspace_bytes < need)) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    if (g.own_scores)
        scores = reinterpret_cast<float*>(reinterpret_cast<uintptr_t>(p->workspace) + 255 & ~(uintptr_t)255);
    cudaStream_t s = (cudaStream_t)stream;
    st = score_any(p, scores, g.nb_stride, reinterpret_cast<char*>(p->workspace) + own, s);
    if (st != SPOT_OK) return st;
    return run_select(p, scores, g.nb_stride, g.rows_per_seq, g.max_nb, s);
}

extern "C" spot_status spot_score_blocks(const spot_select_params* p, void* stream) {
    SelectGeom g;
    spot_status st = select_geometry(p, &g, true);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t need = prefill_scratch_bytes(p);        // quantised cache in prefill: the one case that needs the workspace
    if (need && (!p->workspace || p->workspace_bytes < need)) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    return score_any(p, p->block_scores, g.nb_stride, p->workspace, s);
}

extern "C" spot_status spot_decode_step_host(const spot_decode_step_host_params* p, void* stream) {
    if (!p || !p->sel_q_host || !p->w_host || !p->q_host || !p->out_host || !p->budgets_host) return SPOT_ERR_INVALID_ARG;
    const spot_select_params& sp = p->select;
    const spot_attn_params& ap = p->attn;
    if (sp.q_block != 1 || sp.B != ap.B) return SPOT_ERR_INVALID_ARG;
    // every argument check of the two calls runs before the first copy is enqueued
    {
        SelectGeom g;
        spot_status st0 = select_geometry(&sp, &g);
        if (st0 != SPOT_OK) return st0;
        if ((st0 = check_attn_decode_args(&ap)) != SPOT_OK) return st0;
        if ((st0 = check_device()) != SPOT_OK) return st0;
        // the *_host buffers must be page-locked: a pageable cudaMemcpyAsync blocks the host and cannot be captured
        const void* hosts[5] = {p->sel_q_host, p->w_host, p->q_host, p->out_host, p->budgets_host};
        for (const void* h : hosts) {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, h) != cudaSuccess) { cudaGetLastError(); return SPOT_ERR_INVALID_ARG; }
            if (at.type != cudaMemoryTypeHost && at.type != cudaMemoryTypeManaged) return SPOT_ERR_INVALID_ARG;
        }
    }
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n_selq = (size_t)sp.B * sp.H_idx * sp.d_idx * 2, n_w = (size_t)sp.B * sp.H_idx * 4;
    const size_t n_q = (size_t)ap.B * ap.H_q * ap.D * 2;
    // every small copy costs a few microseconds of stream time: inputs laid out back to back on both sides
    // (sel_q | w | q) go up as one transfer
    const char* h0 = reinterpret_cast<const char*>(p->sel_q_host);
    const char* d0 = reinterpret_cast<const char*>(sp.sel_q);
    const bool in_packed = reinterpret_cast<const char*>(p->w_host) == h0 + n_selq &&
                           reinterpret_cast<const char*>(p->q_host) == h0 + n_selq + n_w &&
                           reinterpret_cast<const char*>(sp.w) == d0 + n_selq &&
                           reinterpret_cast<const char*>(ap.q) == d0 + n_selq + n_w;
    if (in_packed) {
        SPOT_CUDA_TRY(cudaMemcpyAsync((void*)sp.sel_q, p->sel_q_host, n_selq + n_w + n_q, cudaMemcpyHostToDevice, s));
    } else {
        SPOT_CUDA_TRY(cudaMemcpyAsync((void*)sp.sel_q, p->sel_q_host, n_selq, cudaMemcpyHostToDevice, s));
        SPOT_CUDA_TRY(cudaMemcpyAsync((void*)sp.w, p->w_host, n_w, cudaMemcpyHostToDevice, s));
        SPOT_CUDA_TRY(cudaMemcpyAsync((void*)ap.q, p->q_host, n_q, cudaMemcpyHostToDevice, s));
    }
    spot_status st = spot_select(&sp, stream);
    if (st != SPOT_OK) return st;
    st = spot_sparse_attn_decode(&ap, stream);
    if (st != SPOT_OK) return st;
    const size_t n_out = (size_t)ap.B * ap.H_q * ap.D * 2, n_bud = (size_t)sp.B * 4;
    const bool out_packed = reinterpret_cast<char*>(p->budgets_host) == reinterpret_cast<char*>(p->out_host) + n_out &&
                            reinterpret_cast<char*>(sp.budgets) == reinterpret_cast<char*>(ap.out) + n_out;
    if (out_packed) {
        SPOT_CUDA_TRY(cudaMemcpyAsync(p->out_host, ap.out, n_out + n_bud, cudaMemcpyDeviceToHost, s));
    } else {
        SPOT_CUDA_TRY(cudaMemcpyAsync(p->out_host, ap.out, n_out, cudaMemcpyDeviceToHost, s));
        SPOT_CUDA_TRY(cudaMemcpyAsync(p->budgets_host, sp.budgets, n_bud, cudaMemcpyDeviceToHost, s));
    }
    return SPOT_OK;
}
