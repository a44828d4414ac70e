// C-ABI glue: status strings, device check, spot_select orchestration (score kernel -> selection kernel) and the
// host-buffer decode step.  All argument validation happens here, on the host, before any launch.
#include "common.cuh"

#include <chrono>
#include <string.h>

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
spot_status score_decode(const spot_select_params* p, float* scores, int nb_stride, const StepSync* sync, int reserve_sms,
                         cudaStream_t s);
spot_status score_prefill(const spot_select_params* p, float* scores, int nb_stride, int q_fmt, cudaStream_t s);
spot_status run_select(const spot_select_params* p, const float* scores, int nb_stride, int rows_per_seq, int max_nb,
                       const StepSync* sync, cudaStream_t s);
spot_status attn_decode_piped(const spot_attn_params* p, const StepSync* sync, cudaStream_t s);     // attn_decode.cu
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
    if (!selk_is_format(p->fmt)) return SPOT_ERR_INVALID_ARG;
    if (p->mode != SPOT_MODE_TOPK && p->mode != SPOT_MODE_DUAL_TOPP) return SPOT_ERR_INVALID_ARG;
    if (p->B <= 0 || p->Tq <= 0 || p->H_idx <= 0 || p->d_idx <= 0 || p->d_idx % 32 != 0) return SPOT_ERR_INVALID_ARG;
    if (p->blk <= 0 || (!score_only && p->cap <= 0) || p->cache_stride_tokens <= 0) return SPOT_ERR_INVALID_ARG;
    if (p->sink_blocks < 0 || p->recency_blocks < 0 || p->kmin_blocks < 0 || p->top_k < 0) return SPOT_ERR_INVALID_ARG;
    if (p->mode == SPOT_MODE_DUAL_TOPP && !(p->p > 0.0 && p->p <= 1.0)) return SPOT_ERR_INVALID_ARG;
    if (!(p->temperature > 0.0)) return SPOT_ERR_INVALID_ARG;
    if (p->mode == SPOT_MODE_TOPK && p->top_k < p->sink_blocks + p->recency_blocks) return SPOT_ERR_INVALID_ARG;
    if (p->fmt != SPOT_SELK_BF16 && p->cache_stride_tokens % SELK_TILE != 0)
        return SPOT_ERR_INVALID_ARG;
    // quantised selector queries on the tensor cores (f2): FP8-E4M3 queries against the FP8-E4M3 cache, prefill rows only
    // (and, round 2, MXFP4 queries -- a cache of Tq tokens per sequence -- against the MXFP4 cache, block-scaled)
    if (p->q_fmt != SPOT_SELK_BF16 && p->q_fmt != SPOT_SELK_FP8_E4M3 && p->q_fmt != SPOT_SELK_MXFP4) return SPOT_ERR_INVALID_ARG;
    if (p->q_fmt != SPOT_SELK_BF16 && (p->fmt != p->q_fmt || p->q_block != 64)) return SPOT_ERR_UNSUPPORTED;
    // INT4 with BF16 group scales: its keys q * s are not BF16 numbers (R39), and the prefill form would score their
    // dequantised BF16 view -- decode rows only
    if (p->fmt == SPOT_SELK_INT4_BF16S && p->q_block != 1) return SPOT_ERR_UNSUPPORTED;
    // 64-token blocks, or the paper's own 16-token blocks (f3), in both row forms
    if (p->blk != 64 && p->blk != 16) return SPOT_ERR_UNSUPPORTED;
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
    if (p->q_block == 1 || p->fmt == SPOT_SELK_BF16 || p->q_fmt != SPOT_SELK_BF16) return 0;
    return 256 + (size_t)p->B * ((size_t)p->q_start + p->Tq) * p->H_idx * p->d_idx * 2;
}

#ifdef SPOT_TRACE
unsigned long long* g_trace = nullptr;     // development builds only: where the kernels of a step stamp %globaltimer
#endif

// a token unlike the previous call's on the same workspace (common.cuh, StepSync): host clock in ns, salted per thread
unsigned long long fresh_token() {
    static thread_local unsigned long long salt = 0;
    const unsigned long long ns =
        (unsigned long long)std::chrono::steady_clock::now().time_since_epoch().count();
    return ((ns << 8) ^ (++salt & 0xffull)) | 1ull;
}

// the hand-off words of a pipelined call (common.cuh, StepSync): ready[B] laid over `area` (nullptr: no ready words)
StepSync make_sync(void* area, bool with_ready) {
    StepSync y;
    memset(&y, 0, sizeof(y));
    const unsigned long long t = fresh_token();
    y.tag = (uint32_t)(t ^ (t >> 32)) | 1u;
    y.ready = with_ready ? reinterpret_cast<uint32_t*>((reinterpret_cast<uintptr_t>(area) + 63) & ~(uintptr_t)63) : nullptr;
#ifdef SPOT_TRACE
    y.trace = g_trace;
#endif
    return y;
}
size_t sync_area_bytes(int B) { return 64 + step_sync_bytes(B); }   // 64: alignment slack

// decode rows of spot_select / spot_decode_step: the scoring kernel hands its block scores over as 64-bit tagged words
int tagged_stride(const SelectGeom& g) { return (g.max_nb + 3) & ~3; }
size_t tagged_bytes(const spot_select_params* p, const SelectGeom& g) { return (size_t)p->B * tagged_stride(g) * 8; }

// SMs the scoring grid leaves to the selection CTAs that run beside it
int reserve_for_select(int B) { return B < 8 ? B : 8; }

spot_status score_any(const spot_select_params* p, float* scores, int nb_stride, void* scratch_area, const StepSync* sync,
                      cudaStream_t s) {
    if (p->q_block == 1) return score_decode(p, scores, nb_stride, sync, sync ? reserve_for_select(p->B) : 0, s);
    // FP8 x FP8 / MXFP4 x MXFP4: straight from the cache layouts, no dequantise pass
    if (p->q_fmt == SPOT_SELK_FP8_E4M3 || p->q_fmt == SPOT_SELK_MXFP4) return score_prefill(p, scores, nb_stride, p->q_fmt, s);
    if (p->fmt == SPOT_SELK_BF16) return score_prefill(p, scores, nb_stride, SPOT_SELK_BF16, s);
    uint16_t* deq = reinterpret_cast<uint16_t*>((reinterpret_cast<uintptr_t>(scratch_area) + 255) & ~(uintptr_t)255);
    const int tok = p->q_start + p->Tq;
    spot_status st = spot_dequantize_selector_k(p->sel_k, deq, (spot_selk_format)p->fmt, p->B, tok, 0, p->cache_stride_tokens, p->H_idx,
                                                p->d_idx, (void*)s);
    if (st != SPOT_OK) return st;
    spot_select_params q = *p;
    q.sel_k = deq; q.fmt = SPOT_SELK_BF16; q.cache_stride_tokens = tok;
    return score_prefill(&q, scores, nb_stride, SPOT_SELK_BF16, s);
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
extern "C" const char* spot_version(void) { return "0.3"; }   // 0.3: SPOT_SELK_MXINT8 / _INT4_BF16S, q_fmt = MXFP4
extern "C" size_t spot_struct_size(int which) {
    switch (which) {
        case 0: return sizeof(spot_select_params);
        case 1: return sizeof(spot_attn_params);
        case 2: return sizeof(spot_decode_step_host_params);
        case 3: return sizeof(spot_project_params);
        case 4: return sizeof(spot_decode_step_params);
        case 5: return sizeof(spot_train_params);
    }
    return 0;
}

extern "C" size_t spot_select_workspace_bytes(const spot_select_params* p) {
    SelectGeom g;
    // a block without an index list is a spot_score_blocks block (it ignores indices / budgets / cap): size it as such
    if (!p || select_geometry(p, &g, /*score_only=*/!p->indices) != SPOT_OK) return 0;
    size_t bytes = 256;
    if (p->q_block == 1 && p->indices) bytes += tagged_bytes(p, g);          // decode rows: block scores as tagged words
    else if (g.own_scores) bytes += (size_t)p->B * g.rows_per_seq * g.nb_stride * sizeof(float);
    return bytes + prefill_scratch_bytes(p);
}

namespace spot {
namespace {

// a1 + a2.  ext: the hand-offs of a whole step (spot_decode_step; its `ready` words are what the attention kernel waits
// for); nullptr: the call's own, in its workspace, when the rows are decode rows.
spot_status select_impl(const spot_select_params* p, const StepSync* ext, cudaStream_t s) {
    SelectGeom g;
    spot_status st = select_geometry(p, &g);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    const bool piped = p->q_block == 1;
    float* scores = p->block_scores;
    int stride = g.nb_stride;
    size_t own = 0;
    if (piped) { own = 256 + tagged_bytes(p, g); stride = tagged_stride(g); }
    else if (g.own_scores) own = 256 + (size_t)p->B * g.rows_per_seq * g.nb_stride * sizeof(float);
    const size_t need = own + prefill_scratch_bytes(p);
    if (need && (!p->workspace || p->workspace_bytes < need)) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    if (own) scores = reinterpret_cast<float*>(reinterpret_cast<uintptr_t>(p->workspace) + 255 & ~(uintptr_t)255);
    StepSync mine;
    const StepSync* sync = nullptr;
    if (piped) {
        if (ext) sync = ext;
        else { mine = make_sync(nullptr, false); sync = &mine; }
    }
    st = score_any(p, scores, stride, reinterpret_cast<char*>(p->workspace) + own, sync, s);
    if (st != SPOT_OK) return st;
    return run_select(p, scores, stride, g.rows_per_seq, g.max_nb, sync, s);
}

}  // namespace
}  // namespace spot

extern "C" spot_status spot_select(const spot_select_params* p, void* stream) {
    return select_impl(p, nullptr, (cudaStream_t)stream);
}

extern "C" spot_status spot_score_blocks(const spot_select_params* p, void* stream) {
    SelectGeom g;
    spot_status st = select_geometry(p, &g, true);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t need = prefill_scratch_bytes(p);        // quantised cache in prefill: the one case that needs the workspace
    if (need && (!p->workspace || p->workspace_bytes < need)) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    return score_any(p, p->block_scores, g.nb_stride, p->workspace, nullptr, s);
}

namespace spot {
namespace {

// the two parameter blocks of a step must describe ONE step: same batch, same lists, same lengths
spot_status check_step(const spot_select_params& sp, const spot_attn_params& ap) {
    SelectGeom g;
    spot_status st = select_geometry(&sp, &g);
    if (st != SPOT_OK) return st;
    if ((st = check_attn_decode_args(&ap)) != SPOT_OK) return st;
    if (sp.q_block != 1 || sp.B != ap.B || sp.blk != ap.blk) return SPOT_ERR_INVALID_ARG;
    if (ap.indices != sp.indices || ap.budgets != sp.budgets || ap.cap != sp.cap) return SPOT_ERR_INVALID_ARG;
    if (ap.seq_len != sp.seq_len || ap.max_seq_len != sp.max_seq_len) return SPOT_ERR_INVALID_ARG;
    return SPOT_OK;
}

spot_status step_impl(const spot_select_params& sp, const spot_attn_params& ap, void* ws, size_t ws_bytes, cudaStream_t s) {
    if (!ws || ws_bytes < sync_area_bytes(sp.B)) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    const StepSync sync = make_sync(ws, true);
    spot_status st = select_impl(&sp, &sync, s);
    if (st != SPOT_OK) return st;
    return attn_decode_piped(&ap, &sync, s);
}

}  // namespace
}  // namespace spot

extern "C" size_t spot_decode_step_workspace_bytes(const spot_decode_step_params* p) {
    if (!p || check_step(p->select, p->attn) != SPOT_OK) return 0;
    return sync_area_bytes(p->select.B);
}

extern "C" spot_status spot_decode_step(const spot_decode_step_params* p, void* stream) {
    if (!p) return SPOT_ERR_INVALID_ARG;
    spot_status st = check_step(p->select, p->attn);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    return step_impl(p->select, p->attn, p->workspace, p->workspace_bytes, (cudaStream_t)stream);
}

extern "C" spot_status spot_decode_step_host(const spot_decode_step_host_params* p, void* stream) {
    if (!p || !p->sel_q_host || !p->w_host || !p->q_host || !p->out_host || !p->budgets_host) return SPOT_ERR_INVALID_ARG;
    const spot_select_params& sp = p->select;
    const spot_attn_params& ap = p->attn;
    // every argument check of the step runs before the first copy is enqueued
    {
        spot_status st0 = check_step(sp, ap);
        if (st0 != SPOT_OK) return st0;
        if (!p->step_workspace || p->step_workspace_bytes < sync_area_bytes(sp.B)) return SPOT_ERR_WORKSPACE_TOO_SMALL;
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
    spot_status st = step_impl(sp, ap, p->step_workspace, p->step_workspace_bytes, s);
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

#ifdef SPOT_TRACE
extern "C" void spot_debug_set_trace(void* dev_buf) { spot::g_trace = (unsigned long long*)dev_buf; }
#endif
