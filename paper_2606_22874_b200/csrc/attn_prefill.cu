// Step a3' -- block-sparse causal GQA flash attention for chunked prefill (Fig. 2):
// every 64-token query block attends to its own list of selected 64-token key blocks; only the diagonal block needs a
// token-level mask (t <= own position).
//
// Tensor-bound (each 32 KiB K+V tile is reused by 64 queries x G heads).  Work item = (sequence, query block, KV head,
// 128-row tile): the 64 queries x G query heads of the group are stacked as rows, row = head_in_group * 64 + query, so
// one K/V tile in shared memory feeds every head of the group.  8 warps x 16 rows; K/V tiles arrive through a
// 3-stage cp.async ring (XOR-swizzled 256-byte rows, conflict-free ldmatrix); S = Q K^T and O += P V run on
// mma.sync m16n8k16 with fp32 accumulation and a register-resident online softmax (log2 domain).
// This is the first, parity-checked form of the step; the tcgen05/TMEM form is DESIGN.md section 8's next item.
#include "common.cuh"

namespace spot {

namespace {

constexpr bool PA_USE_TCGEN05 = true;           // attn_prefill_tc.cu; the mma.sync kernel below is the first form
constexpr int PA_WARPS = 8;
constexpr int PA_ROWS = PA_WARPS * 16;          // 128 rows per CTA
constexpr int PA_STAGES = 3;
constexpr int PA_D = 128;
constexpr int PA_TILE_BYTES = 64 * PA_D * 2;    // 16 KiB (K or V block of one head)
constexpr int PA_STAGE_BYTES = 2 * PA_TILE_BYTES;
constexpr int PA_SMEM = PA_STAGES * PA_STAGE_BYTES;   // 96 KiB

struct PrefillAttnArgs {
    const uint16_t* q;           // [B][Tq][H_q][128]
    const uint16_t* k;
    const uint16_t* v;
    int64_t sb, st, sh;          // element strides: batch, token, head
    const int32_t* indices;      // [B * n_qb][cap]; nullptr: every causally visible block
    const int32_t* budgets;
    int cap;
    int Tq, n_qb, H_q, H_kv, G;
    int qb_start;                // q_start / 64
    float scale_log2;
    uint16_t* out;               // [B][Tq][H_q][128]
    float* lse;                  // optional [B][Tq][H_q]
};

__device__ __forceinline__ uint32_t pa_sw(int row, int chunk) { return (uint32_t)(row * 256 + ((chunk ^ (row & 7)) << 4)); }

// one 64 x 128 BF16 tile (rows `st` elements apart) -> swizzled smem; 256 threads x 4 chunks of 16 B
__device__ __forceinline__ void pa_issue_tile(uint32_t smem_tile, const uint16_t* base, int64_t st, int tid) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int id = i * (PA_WARPS * 32) + tid;
        const int row = id >> 4, ch = id & 15;
        cp_async16(smem_tile + pa_sw(row, ch), base + (int64_t)row * st + ch * 8, true);
    }
}

__global__ void __launch_bounds__(PA_WARPS * 32, 1) attn_prefill_kernel(PrefillAttnArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int mt = blockIdx.x, hk = blockIdx.y;
    const int rowz = (int)gridDim.z - 1 - (int)blockIdx.z;      // heaviest (latest) query blocks are scheduled first
    const int b = rowz / a.n_qb, i = rowz - b * a.n_qb;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, c = lane & 3;
    const int G = a.G;
    const int qb_abs = a.qb_start + i;                           // the query block's own (diagonal) key block
    const int budget = a.indices ? min(a.budgets[rowz], a.cap) : qb_abs + 1;
    const int32_t* idx = a.indices ? a.indices + (int64_t)rowz * a.cap : nullptr;

    // rows of this warp: tile rows 16 warp .. +15; row -> (head in group, query in block); a warp's rows share a head
    const int row0 = mt * PA_ROWS + warp * 16;
    const int hg = row0 >> 6;                                    // head in group
    const bool warp_live = hg < G;
    const int ql0 = (row0 & 63) + g, ql1 = ql0 + 8;              // the two query rows of this lane (within the block)
    const int h = hk * G + hg;

    // Q fragments (A operand)
    uint32_t qa[8][4];
    {
        const uint16_t* q0 = a.q + (((int64_t)b * a.Tq + i * 64 + ql0) * a.H_q + h) * PA_D;
        const uint16_t* q1 = a.q + (((int64_t)b * a.Tq + i * 64 + ql1) * a.H_q + h) * PA_D;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const int col = ks * 16 + c * 2;
            qa[ks][0] = warp_live ? *reinterpret_cast<const uint32_t*>(q0 + col) : 0u;
            qa[ks][1] = warp_live ? *reinterpret_cast<const uint32_t*>(q1 + col) : 0u;
            qa[ks][2] = warp_live ? *reinterpret_cast<const uint32_t*>(q0 + col + 8) : 0u;
            qa[ks][3] = warp_live ? *reinterpret_cast<const uint32_t*>(q1 + col + 8) : 0u;
        }
    }

    const uint16_t* kbase = a.k + (int64_t)b * a.sb + (int64_t)hk * a.sh;
    const uint16_t* vbase = a.v + (int64_t)b * a.sb + (int64_t)hk * a.sh;
    const uint32_t smem0 = smem_u32(smem);

    float o[16][4];
#pragma unroll
    for (int n = 0; n < 16; ++n) o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f;
    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;

    auto block_of = [&](int it) -> int { return idx ? idx[it] : it; };
    auto issue = [&](int it) {
        const int j = block_of(it);
        // blocks past the diagonal are never visible; they are skipped at compute time, load a valid tile anyway
        const int jl = min(max(j, 0), qb_abs);
        const uint32_t sbase = smem0 + (it % PA_STAGES) * PA_STAGE_BYTES;
        pa_issue_tile(sbase, kbase + (int64_t)jl * 64 * a.st, a.st, tid);
        pa_issue_tile(sbase + PA_TILE_BYTES, vbase + (int64_t)jl * 64 * a.st, a.st, tid);
    };

#pragma unroll
    for (int s = 0; s < PA_STAGES - 1; ++s) {
        if (s < budget) issue(s);
        cp_async_commit();
    }

    for (int it = 0; it < budget; ++it) {
        cp_async_wait<PA_STAGES - 2>();
        __syncthreads();                       // tile `it` has landed for everyone; stage (it-1)%S is free again
        {
            const int nx = it + PA_STAGES - 1;
            if (nx < budget) issue(nx);
            cp_async_commit();
        }
        const int j = block_of(it);
        if (j < 0 || j > qb_abs || !warp_live) continue;          // CTA-uniform except warp_live (warp-uniform)
        const uint32_t ks_base = smem0 + (it % PA_STAGES) * PA_STAGE_BYTES;
        const uint32_t vs_base = ks_base + PA_TILE_BYTES;

        // S = Q K^T : 16 rows x 64 tokens
        float s[8][4];
#pragma unroll
        for (int n = 0; n < 8; ++n) s[n][0] = s[n][1] = s[n][2] = s[n][3] = 0.f;
        {
            const int mi = lane >> 3, r8 = lane & 7;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
#pragma unroll
                for (int tg = 0; tg < 4; ++tg) {
                    const int row = tg * 16 + (mi >> 1) * 8 + r8;
                    uint32_t b0, b1, b2, b3;
                    ldmatrix_x4(b0, b1, b2, b3, ks_base + pa_sw(row, 2 * ks + (mi & 1)));
                    mma_bf16_16816(s[2 * tg], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b0, b1);
                    mma_bf16_16816(s[2 * tg + 1], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b2, b3);
                }
            }
        }
        const bool diag = (j == qb_abs);
#pragma unroll
        for (int n = 0; n < 8; ++n)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int t = n * 8 + c * 2 + (e & 1);
                const int ql = (e & 2) ? ql1 : ql0;
                s[n][e] = (diag && t > ql) ? -INFINITY : s[n][e] * a.scale_log2;
            }
        float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            mx0 = fmaxf(mx0, fmaxf(s[n][0], s[n][1]));
            mx1 = fmaxf(mx1, fmaxf(s[n][2], s[n][3]));
        }
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
        mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
        mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
        const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
        const float mu0 = (mn0 == -INFINITY) ? 0.f : mn0, mu1 = (mn1 == -INFINITY) ? 0.f : mn1;
        const float c0 = fast_exp2(m0 - mu0), c1 = fast_exp2(m1 - mu1);
        m0 = mn0; m1 = mn1;
        float ps0 = 0.f, ps1 = 0.f;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            s[n][0] = fast_exp2(s[n][0] - mu0); s[n][1] = fast_exp2(s[n][1] - mu0);
            s[n][2] = fast_exp2(s[n][2] - mu1); s[n][3] = fast_exp2(s[n][3] - mu1);
            ps0 += s[n][0] + s[n][1];
            ps1 += s[n][2] + s[n][3];
        }
        l0 = l0 * c0 + ps0;
        l1 = l1 * c1 + ps1;
#pragma unroll
        for (int n = 0; n < 16; ++n) { o[n][0] *= c0; o[n][1] *= c0; o[n][2] *= c1; o[n][3] *= c1; }

        // O += P V
        {
            const int mi = lane >> 3, r8 = lane & 7;
#pragma unroll
            for (int kt = 0; kt < 4; ++kt) {
                const uint32_t pa0 = pack_bf16x2(s[2 * kt][0], s[2 * kt][1]), pa1 = pack_bf16x2(s[2 * kt][2], s[2 * kt][3]);
                const uint32_t pa2 = pack_bf16x2(s[2 * kt + 1][0], s[2 * kt + 1][1]);
                const uint32_t pa3 = pack_bf16x2(s[2 * kt + 1][2], s[2 * kt + 1][3]);
                const int row = kt * 16 + (mi & 1) * 8 + r8;
#pragma unroll
                for (int nd = 0; nd < 16; nd += 2) {
                    uint32_t b0, b1, b2, b3;
                    ldmatrix_x4_trans(b0, b1, b2, b3, vs_base + pa_sw(row, nd + (mi >> 1)));
                    mma_bf16_16816(o[nd], pa0, pa1, pa2, pa3, b0, b1);
                    mma_bf16_16816(o[nd + 1], pa0, pa1, pa2, pa3, b2, b3);
                }
            }
        }
    }
    cp_async_wait<0>();
    if (!warp_live) return;

    l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
    const float r0 = l0 > 0.f ? 1.f / l0 : 0.f, r1 = l1 > 0.f ? 1.f / l1 : 0.f;
    uint16_t* o0 = a.out + (((int64_t)b * a.Tq + i * 64 + ql0) * a.H_q + h) * PA_D;
    uint16_t* o1 = a.out + (((int64_t)b * a.Tq + i * 64 + ql1) * a.H_q + h) * PA_D;
#pragma unroll
    for (int n = 0; n < 16; ++n) {
        const int col = n * 8 + c * 2;
        *reinterpret_cast<uint32_t*>(o0 + col) = pack_bf16x2(o[n][0] * r0, o[n][1] * r0);
        *reinterpret_cast<uint32_t*>(o1 + col) = pack_bf16x2(o[n][2] * r1, o[n][3] * r1);
    }
    if (a.lse && c == 0) {
        a.lse[((int64_t)b * a.Tq + i * 64 + ql0) * a.H_q + h] = l0 > 0.f ? (m0 + log2f(l0)) * 0.6931471805599453f : -INFINITY;
        a.lse[((int64_t)b * a.Tq + i * 64 + ql1) * a.H_q + h] = l1 > 0.f ? (m1 + log2f(l1)) * 0.6931471805599453f : -INFINITY;
    }
}

spot_status check_prefill(const spot_attn_params* p) {
    if (!p || !p->q || !p->k || !p->v || !p->out) return SPOT_ERR_INVALID_ARG;
    if (!aligned16(p->q) || !aligned16(p->k) || !aligned16(p->v) || !aligned16(p->out)) return SPOT_ERR_INVALID_ARG;
    if (p->B <= 0 || p->H_q <= 0 || p->H_kv <= 0 || p->H_q % p->H_kv != 0) return SPOT_ERR_INVALID_ARG;
    if (p->Tq <= 0 || p->Tq % 64 != 0 || p->q_start < 0 || p->q_start % 64 != 0) return SPOT_ERR_INVALID_ARG;   // R26
    if (p->H_q / p->H_kv > 16) return SPOT_ERR_UNSUPPORTED;
    if (p->D != 128 || p->blk != 64) return SPOT_ERR_UNSUPPORTED;
    if (p->kv_stride_token < p->D || p->kv_stride_token % 8 || p->kv_stride_head % 8 || p->kv_stride_batch % 8)
        return SPOT_ERR_INVALID_ARG;
    if (p->indices && (!p->budgets || p->cap <= 0)) return SPOT_ERR_INVALID_ARG;
    if ((int64_t)p->B * (p->Tq / 64) > 65535) return SPOT_ERR_UNSUPPORTED;
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
    if (PA_USE_TCGEN05) return attn_prefill_tc(p, (cudaStream_t)stream);
    PrefillAttnArgs a;
    a.q = p->q; a.k = p->k; a.v = p->v;
    a.sb = p->kv_stride_batch; a.st = p->kv_stride_token; a.sh = p->kv_stride_head;
    a.indices = p->indices; a.budgets = p->budgets; a.cap = p->cap;
    a.Tq = p->Tq; a.n_qb = p->Tq / 64; a.H_q = p->H_q; a.H_kv = p->H_kv; a.G = p->H_q / p->H_kv;
    a.qb_start = p->q_start / 64;
    a.scale_log2 = p->sm_scale * 1.4426950408889634f;
    a.out = p->out; a.lse = p->lse;
    static bool attr_set = false;
    if (!attr_set) {
        SPOT_CUDA_TRY(cudaFuncSetAttribute(attn_prefill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PA_SMEM));
        attr_set = true;
    }
    const int n_mt = (a.G * 64 + PA_ROWS - 1) / PA_ROWS;
    dim3 grid((unsigned)n_mt, (unsigned)p->H_kv, (unsigned)(p->B * a.n_qb));
    attn_prefill_kernel<<<grid, PA_WARPS * 32, PA_SMEM, (cudaStream_t)stream>>>(a);
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}
