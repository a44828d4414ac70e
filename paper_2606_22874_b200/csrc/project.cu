// Step f1 (the step right before the path) -- selector projections, RoPE and mixing weights for
// the current token of every sequence, and the append of its selector key to the cache (
// DESIGN.md readings R27-R29):  q^I = RoPE(W_q h), k^I = RoPE(W_k h), w = W_w h.
//
// A matrix-vector product shared by the B sequences of the step: (2 H d + H) x d_model BF16 weights (4.2 MiB at
// 4 x 64 x 4096) are read once -- HBM-bound, ~1 us of traffic, so the kernel is shaped for latency: one CTA per PAIR
// of output rows (the two rows a rotary pair needs, so the rotation happens in registers), its four warps splitting
// d_model, eight 16-byte weight loads in flight per thread before the first FMA, fp32 FMAs, butterfly + shared-memory
// reduction, fp64 sincos for the angle (positions reach 2^17).
// The new k^I goes to a small BF16 staging row and is appended by quantize.cu's kernels in the cache's own format
// (programmatic dependent launch), so that a0's bit-exact quantiser definition has a single implementation.
#include <math.h>

#include "common.cuh"

namespace spot {

spot_status append_selector_k(const uint16_t* k_new, void* cache, int fmt, int B, const int32_t* pos, int64_t stride,
                              int H, int d, cudaStream_t s);     // quantize.cu

namespace {

constexpr int PJ_WARPS = 4;
constexpr int PJ_BC = 8;            // sequences per pass over a pair of weight rows
constexpr int PJ_MAX_ROPE = 256;

struct ProjectArgs {
    const uint16_t* hidden;
    const uint16_t* w_q;
    const uint16_t* w_k;
    const uint16_t* w_w;
    const int32_t* pos;
    int B, d_model, H, d, rope;
    float rope_base;
    uint16_t* sel_q;
    uint16_t* k_new;      // staging [B][H*d] BF16
    float* w;
    int n_qk_units;       // H*d/2 pair units per projection
    int n_units;          // 2 * n_qk_units + ceil(H/2)
    double inv_freq[PJ_MAX_ROPE / 2];   // base^(-2 i / rope), computed on the host in fp64 (keeps pow() off the device path)
};

__device__ __forceinline__ float dot8(uint4 a, uint4 b, float acc) {
    acc = fmaf(bf16lo(a.x), bf16lo(b.x), acc); acc = fmaf(bf16hi(a.x), bf16hi(b.x), acc);
    acc = fmaf(bf16lo(a.y), bf16lo(b.y), acc); acc = fmaf(bf16hi(a.y), bf16hi(b.y), acc);
    acc = fmaf(bf16lo(a.z), bf16lo(b.z), acc); acc = fmaf(bf16hi(a.z), bf16hi(b.z), acc);
    acc = fmaf(bf16lo(a.w), bf16lo(b.w), acc); acc = fmaf(bf16hi(a.w), bf16hi(b.w), acc);
    return acc;
}

__global__ void __launch_bounds__(PJ_WARPS * 32) project_rope_kernel(ProjectArgs a) {
    __shared__ float part[PJ_WARPS][2 * PJ_BC];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int unit = blockIdx.x;                     // one CTA per pair of output rows; its 4 warps split d_model
    pdl_wait();
    pdl_launch_dependents();
    // unit -> (matrix, two output rows, rotary pair index or -1)
    const uint16_t* W;
    int r0, r1, pair_i = -1, kind;                   // kind 0: q, 1: k, 2: w
    if (unit < 2 * a.n_qk_units) {
        kind = unit / a.n_qk_units;
        const int p = unit - kind * a.n_qk_units;
        const int head = p / (a.d / 2), ii = p - head * (a.d / 2);
        W = kind ? a.w_k : a.w_q;
        if (ii < a.rope / 2) { r0 = head * a.d + ii; r1 = r0 + a.rope / 2; pair_i = ii; }
        else { r0 = head * a.d + a.rope + 2 * (ii - a.rope / 2); r1 = r0 + 1; }
    } else {
        kind = 2;
        W = a.w_w;
        r0 = 2 * (unit - 2 * a.n_qk_units);
        r1 = min(r0 + 1, a.H - 1);
    }
    const uint4* w0 = reinterpret_cast<const uint4*>(W + (int64_t)r0 * a.d_model);
    const uint4* w1 = reinterpret_cast<const uint4*>(W + (int64_t)r1 * a.d_model);
    const int n_vec = a.d_model / 8;                 // 16-byte vectors per row; a multiple of 32

    for (int b0 = 0; b0 < a.B; b0 += PJ_BC) {
        float acc0[PJ_BC], acc1[PJ_BC];
#pragma unroll
        for (int j = 0; j < PJ_BC; ++j) acc0[j] = acc1[j] = 0.f;
        // four vectors of each weight row per thread and trip, all eight loads in flight before the first FMA: the
        // kernel is a chain of DRAM latencies, not of bytes
        for (int v0 = tid; v0 < n_vec; v0 += 4 * PJ_WARPS * 32) {
            uint4 xa[4], xb[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int v = v0 + u * PJ_WARPS * 32;
                xa[u] = v < n_vec ? ldg_stream_v4(w0 + v) : make_uint4(0, 0, 0, 0);
                xb[u] = v < n_vec ? ldg_stream_v4(w1 + v) : make_uint4(0, 0, 0, 0);
            }
#pragma unroll
            for (int j = 0; j < PJ_BC; ++j) {
                if (b0 + j < a.B) {
                    const uint4* hp = reinterpret_cast<const uint4*>(a.hidden + (int64_t)(b0 + j) * a.d_model);
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int v = v0 + u * PJ_WARPS * 32;
                        if (v < n_vec) {
                            const uint4 hv = __ldg(hp + v);
                            acc0[j] = dot8(xa[u], hv, acc0[j]);
                            acc1[j] = dot8(xb[u], hv, acc1[j]);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < PJ_BC; ++j)
#pragma unroll
            for (int o = 16; o; o >>= 1) {
                acc0[j] += __shfl_xor_sync(0xffffffffu, acc0[j], o);
                acc1[j] += __shfl_xor_sync(0xffffffffu, acc1[j], o);
            }
        __syncthreads();                             // (the previous pass has read `part`)
        if (lane == 0) {
#pragma unroll
            for (int j = 0; j < PJ_BC; ++j) { part[warp][2 * j] = acc0[j]; part[warp][2 * j + 1] = acc1[j]; }
        }
        __syncthreads();
        // thread j of warp 0 finishes sequence b0 + j
        const int b = b0 + tid;
        if (tid < PJ_BC && b < a.B) {
            float x0 = 0.f, x1 = 0.f;
#pragma unroll
            for (int w = 0; w < PJ_WARPS; ++w) { x0 += part[w][2 * tid]; x1 += part[w][2 * tid + 1]; }
            if (kind == 2) {
                a.w[(int64_t)b * a.H + r0] = x0;
                if (r1 != r0) a.w[(int64_t)b * a.H + r1] = x1;
            } else {
                float y0 = x0, y1 = x1;
                if (pair_i >= 0) {
                    // angle = pos * base^(-2 i / rope); fp64: positions reach 2^17 and the angle must be good to ~1e-7
                    const double ang = (double)a.pos[b] * a.inv_freq[pair_i];
                    double sn, cs;
                    sincos(ang, &sn, &cs);
                    y0 = (float)((double)x0 * cs - (double)x1 * sn);
                    y1 = (float)((double)x1 * cs + (double)x0 * sn);
                }
                uint16_t* dst = (kind ? a.k_new : a.sel_q) + (int64_t)b * a.H * a.d;
                dst[r0] = __bfloat16_as_ushort(__float2bfloat16_rn(y0));
                dst[r1] = __bfloat16_as_ushort(__float2bfloat16_rn(y1));
            }
        }
    }
}

spot_status check_project(const spot_project_params* p) {
    if (!p || !p->hidden || !p->w_q || !p->w_k || !p->w_w || !p->pos || !p->sel_q || !p->w || !p->sel_k)
        return SPOT_ERR_INVALID_ARG;
    if (!aligned16(p->hidden) || !aligned16(p->w_q) || !aligned16(p->w_k) || !aligned16(p->w_w) || !aligned16(p->sel_q) ||
        !aligned16(p->sel_k))
        return SPOT_ERR_INVALID_ARG;
    if (p->B <= 0 || p->H_idx <= 0 || p->d_idx <= 0 || p->d_idx % 32 != 0 || p->d_model <= 0 || p->d_model % 256 != 0)
        return SPOT_ERR_INVALID_ARG;
    if (p->rope_dims < 0 || p->rope_dims % 2 != 0 || p->rope_dims > p->d_idx || !(p->rope_base > 0.f))
        return SPOT_ERR_INVALID_ARG;
    if (p->rope_dims > PJ_MAX_ROPE) return SPOT_ERR_UNSUPPORTED;
    if (!selk_is_format(p->fmt)) return SPOT_ERR_INVALID_ARG;
    if (p->cache_stride_tokens <= 0) return SPOT_ERR_INVALID_ARG;
    if (p->fmt != SPOT_SELK_BF16 && p->cache_stride_tokens % SELK_TILE != 0)
        return SPOT_ERR_INVALID_ARG;
    return SPOT_OK;
}

}  // namespace

}  // namespace spot

using namespace spot;

extern "C" size_t spot_selector_project_append_workspace_bytes(const spot_project_params* p) {
    if (check_project(p) != SPOT_OK) return 0;
    return (size_t)p->B * p->H_idx * p->d_idx * 2 + 256;
}

extern "C" spot_status spot_selector_project_append(const spot_project_params* p, void* stream) {
    spot_status st = check_project(p);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    const size_t need = (size_t)p->B * p->H_idx * p->d_idx * 2 + 256;
    if (!p->workspace || p->workspace_bytes < need) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    ProjectArgs a;
    a.hidden = p->hidden; a.w_q = p->w_q; a.w_k = p->w_k; a.w_w = p->w_w; a.pos = p->pos;
    a.B = p->B; a.d_model = p->d_model; a.H = p->H_idx; a.d = p->d_idx; a.rope = p->rope_dims; a.rope_base = p->rope_base;
    a.sel_q = p->sel_q; a.w = p->w;
    a.k_new = reinterpret_cast<uint16_t*>((reinterpret_cast<uintptr_t>(p->workspace) + 255) & ~(uintptr_t)255);
    for (int i = 0; i < p->rope_dims / 2; ++i)
        a.inv_freq[i] = pow((double)p->rope_base, -2.0 * (double)i / (double)p->rope_dims);
    a.n_qk_units = p->H_idx * p->d_idx / 2;
    a.n_units = 2 * a.n_qk_units + (p->H_idx + 1) / 2;
    cudaStream_t s = (cudaStream_t)stream;
    SPOT_CUDA_TRY(launch_pdl(project_rope_kernel, dim3((unsigned)a.n_units), dim3(PJ_WARPS * 32), 0, s, a));
    return append_selector_k(a.k_new, p->sel_k, p->fmt, p->B, p->pos, p->cache_stride_tokens, p->H_idx, p->d_idx, s);
}
