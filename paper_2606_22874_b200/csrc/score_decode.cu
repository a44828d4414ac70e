// Step a1, decode form -- stream the selector K-cache once and emit one score per 64-token block:
//   s[t] = sum_h w_h ReLU(q_h . k_{h,t}),   s_bar[b] = max_{t in b} s[t].
//
// HBM-bound: 512 B (BF16) or 136 B (4-bit) per token, 2 flop/B.  One warp owns one 64-token tile at a time;
// lanes issue 128-bit streaming loads straight into mma.sync A-fragments (no shared-memory staging: there is no
// reuse), the query sits in the B fragment (column 0 only -- the tensor pipe is idle otherwise, so the wasted
// columns are free) and the per-token reduction over d_idx happens inside the MMA instead of in shuffles.
//   BF16 cache : bf16 HMMA, products exact, fp32 accumulate.
//   4-bit cache: codes are unpacked to fp16 pairs in registers (INT4: magic-number OR + one HFMA2 per pair;
//                MXFP4: cvt.rn.f16x2.e2m1x2, one instruction per pair), multiplied against an fp16 copy of the
//                query (pre-scaled per head by a power of two so that the copy is exact for every element
//                within 2^-29 of the head's largest), and the group scale is applied to the 32-element partial
//                sum after the MMA (one FMUL per group instead of one per element).
// The k index of each MMA is a fixed permutation of the d_idx axis applied to both operands, chosen so that
// every lane's 16-byte load lands directly in fragment registers.
#include "common.cuh"

namespace spot {

namespace {

constexpr int SCORE_WARPS = 4;

// four bytes of E2M1 pairs -> four fp16 pairs; the vector mov lets ptxas use F2FP's byte selectors (.B0-.B3),
// one instruction per pair and no shift/mask.
__device__ __forceinline__ void e2m1x8_to_f16x2x4(uint32_t w, uint32_t (&p)[4]) {
    asm("{ .reg .b8 b0, b1, b2, b3; mov.b32 {b0, b1, b2, b3}, %4;\n"
        "cvt.rn.f16x2.e2m1x2 %0, b0; cvt.rn.f16x2.e2m1x2 %1, b1;\n"
        "cvt.rn.f16x2.e2m1x2 %2, b2; cvt.rn.f16x2.e2m1x2 %3, b3; }"
        : "=r"(p[0]), "=r"(p[1]), "=r"(p[2]), "=r"(p[3]) : "r"(w));
}

__device__ __forceinline__ uint32_t hfma2_u32(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t hsub2_u32(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}

// 8 codes (one 32-bit word) -> 4 fp16 pairs; pair pp = dims (2pp, 2pp+1) of the word.
template <int FMT>
__device__ __forceinline__ void unpack8(uint32_t w, uint32_t (&p)[4]) {
    if (FMT == SPOT_SELK_MXFP4) {
        e2m1x8_to_f16x2x4(w, p);
    } else {
        // u = q + 8 in each nibble.  0x6400 | u = 1024 + u (fp16); nibble at bit 4: 1024 + 16 u.
        const uint32_t MAGIC = 0x64006400u;
        const uint32_t C1032 = 0x64086408u;   // 1032.0 x2
        const uint32_t SIXTEENTH = 0x2c002c00u;  // 0.0625 x2
        const uint32_t NEG72 = 0xd480d480u;   // -72.0 x2
        uint32_t w8 = w >> 8;
        p[0] = hsub2_u32((w & 0x000f000fu) | MAGIC, C1032);
        p[1] = hfma2_u32((w & 0x00f000f0u) | MAGIC, SIXTEENTH, NEG72);
        p[2] = hsub2_u32((w8 & 0x000f000fu) | MAGIC, C1032);
        p[3] = hfma2_u32((w8 & 0x00f000f0u) | MAGIC, SIXTEENTH, NEG72);
    }
}

template <int FMT>
__device__ __forceinline__ float scale_to_f32(uint32_t byte) {
    if (FMT == SPOT_SELK_MXFP4) {
        return byte ? __uint_as_float(byte << 23) : __uint_as_float(0x00400000u);
    } else {
        // E4M3 -> fp32 (exact): normal: 2^(E-7)(1+m/8); subnormal: m 2^-9
        uint32_t E = (byte >> 3) & 0xf, m = byte & 7;
        float nrm = __uint_as_float(((E + 120u) << 23) | (m << 20));
        float sub = (float)m * 0.001953125f;
        return E ? nrm : sub;
    }
}

// ---------------------------------------------------------------------------------------------------
// BF16 cache
// ---------------------------------------------------------------------------------------------------
template <int H, int D_IDX>
__global__ void __launch_bounds__(SCORE_WARPS * 32) score_decode_bf16_kernel(
    const uint16_t* __restrict__ sel_q, const float* __restrict__ w, const uint16_t* __restrict__ sel_k,
    int64_t cache_stride_tokens, const int32_t* __restrict__ seq_len, float* __restrict__ scores, int nb_stride) {
    constexpr int ROW = H * D_IDX;          // elements per token
    constexpr int NSEG = ROW / 32;          // 64-byte segments per token
    constexpr int SEG_PER_HEAD = D_IDX / 32;
    const int b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, c = lane & 3;
    pdl_wait();
    pdl_launch_dependents();
    const int L = seq_len[b];
    const int n_b = (L + 63) >> 6;

    // query fragments: only the lanes that hold column 0 of B (g == 0) carry q; k-permutation as in the header.
    uint32_t qf[NSEG][4];
    {
        const uint4* qp = reinterpret_cast<const uint4*>(sel_q + (int64_t)b * ROW);
#pragma unroll
        for (int s = 0; s < NSEG; ++s) {
            uint4 v = make_uint4(0, 0, 0, 0);
            if (g == 0) v = qp[s * 4 + c];
            qf[s][0] = v.x; qf[s][1] = v.y; qf[s][2] = v.z; qf[s][3] = v.w;
        }
    }
    float wh[H];
#pragma unroll
    for (int h = 0; h < H; ++h) wh[h] = w[(int64_t)b * H + h];

    const uint16_t* kb = sel_k + (int64_t)b * cache_stride_tokens * ROW;
    for (int tile = blockIdx.x * SCORE_WARPS + warp; tile < n_b; tile += gridDim.x * SCORE_WARPS) {
        float m = -INFINITY;
        const int t0 = tile * 64;
#pragma unroll 1
        for (int it = 0; it < 4; ++it) {
            const int ta = t0 + it * 16 + g, tb = ta + 8;
            const uint4* ra = reinterpret_cast<const uint4*>(kb + (int64_t)min(ta, L - 1) * ROW) + c;
            const uint4* rb = reinterpret_cast<const uint4*>(kb + (int64_t)min(tb, L - 1) * ROW) + c;
            uint4 va[NSEG], vb[NSEG];
#pragma unroll
            for (int s = 0; s < NSEG; ++s) {
                va[s] = ldg_stream_v4(ra + s * 4);
                vb[s] = ldg_stream_v4(rb + s * 4);
            }
            float sa = 0.f, sb = 0.f;
#pragma unroll
            for (int h = 0; h < H; ++h) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int ss = 0; ss < SEG_PER_HEAD; ++ss) {
                    const int s = h * SEG_PER_HEAD + ss;
                    mma_bf16_16816(acc, va[s].x, vb[s].x, va[s].y, vb[s].y, qf[s][0], qf[s][1]);
                    mma_bf16_16816(acc, va[s].z, vb[s].z, va[s].w, vb[s].w, qf[s][2], qf[s][3]);
                }
                sa = fmaf(wh[h], fmaxf(acc[0], 0.f), sa);   // column 0, row g     (valid on lanes c == 0)
                sb = fmaf(wh[h], fmaxf(acc[2], 0.f), sb);   // column 0, row g + 8
            }
            if (ta < L) m = fmaxf(m, sa);
            if (tb < L) m = fmaxf(m, sb);
        }
        if (c != 0) m = -INFINITY;
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 4));
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 8));
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 16));
        if (lane == 0) scores[(int64_t)b * nb_stride + tile] = m;
    }
}

// ---------------------------------------------------------------------------------------------------
// 4-bit caches (INT4 + E4M3 scale, MXFP4)
// ---------------------------------------------------------------------------------------------------
template <int H, int D_IDX, int FMT>
__global__ void __launch_bounds__(SCORE_WARPS * 32) score_decode_q4_kernel(
    const uint16_t* __restrict__ sel_q, const float* __restrict__ w, const uint8_t* __restrict__ sel_k,
    int64_t tiles_per_seq, const int32_t* __restrict__ seq_len, float* __restrict__ scores, int nb_stride) {
    constexpr int ROW = H * D_IDX;
    constexpr int CPT = ROW / 2;            // code bytes per token
    constexpr int NG = ROW / 32;            // groups (= scale bytes) per token
    constexpr int NQL = NG / 4;             // 64-byte "quad loads" per token: 4 groups, one per lane of a quad
    constexpr int GPH = D_IDX / 32;         // groups per head (2 or 4)
    constexpr int64_t TILE_BYTES = 64 * (CPT + NG);
    static_assert(GPH == 2 || GPH == 4, "d_idx must be 64 or 128 for the 4-bit scoring kernels");
    static_assert(NG % 4 == 0, "H_idx * d_idx must be a multiple of 128");

    __shared__ __align__(16) __half q16[ROW];   // fp16 copy of q, pre-scaled per head by 2^sh[h]
    __shared__ float post[H];                   // 2^-sh[h]

    const int b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, c = lane & 3;
    pdl_wait();
    pdl_launch_dependents();
    const int L = seq_len[b];
    const int n_b = (L + 63) >> 6;

    // prologue: one warp per head finds the head's largest |q| exponent and writes the scaled fp16 copy.
    for (int h = warp; h < H; h += SCORE_WARPS) {
        const uint16_t* qh = sel_q + (int64_t)b * ROW + h * D_IDX;
        float mx = 0.f;
        for (int i = lane; i < D_IDX; i += 32) mx = fmaxf(mx, fabsf(bf16_bits_to_float(qh[i])));
#pragma unroll
        for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        int sh = 0;
        if (mx > 0.f) sh = 14 - ilogbf(mx);       // largest element lands in [2^14, 2^15)
        sh = max(-100, min(100, sh));
        float up = __uint_as_float((uint32_t)(127 + sh) << 23);
        for (int i = lane; i < D_IDX; i += 32) q16[h * D_IDX + i] = __float2half_rn(bf16_bits_to_float(qh[i]) * up);
        if (lane == 0) post[h] = __uint_as_float((uint32_t)(127 - sh) << 23);
    }
    __syncthreads();

    // B fragments: column n of the MMA is the group held by quad-lane c == n; only lane (g == n, c == n) is non-zero.
    uint32_t qf[NQL][16];
#pragma unroll
    for (int ql = 0; ql < NQL; ++ql) {
        const uint4* src = reinterpret_cast<const uint4*>(q16 + (ql * 4 + c) * 32);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            uint4 v = make_uint4(0, 0, 0, 0);
            if (g == c) v = src[i];
            qf[ql][4 * i + 0] = v.x; qf[ql][4 * i + 1] = v.y; qf[ql][4 * i + 2] = v.z; qf[ql][4 * i + 3] = v.w;
        }
    }
    // lanes c < 2 read columns 2c, 2c+1 = groups 4ql + 2c (+1); their head, weight and power-of-two post-scale:
    float wq[NQL], ps[NQL];
#pragma unroll
    for (int ql = 0; ql < NQL; ++ql) {
        int head = (4 * ql + 2 * (c & 1)) / GPH;
        wq[ql] = w[(int64_t)b * H + head];
        ps[ql] = post[head];
    }

    const uint8_t* kb = sel_k + (int64_t)b * tiles_per_seq * TILE_BYTES;
    for (int tile = blockIdx.x * SCORE_WARPS + warp; tile < n_b; tile += gridDim.x * SCORE_WARPS) {
        const uint8_t* tb = kb + (int64_t)tile * TILE_BYTES;
        const int t0 = tile * 64;
        // whole tile in flight: 16 x LDG.128 of codes per lane (8 KiB per warp) + the scale bytes
        uint4 cd[4][NQL][2];
#pragma unroll
        for (int it = 0; it < 4; ++it)
#pragma unroll
            for (int ql = 0; ql < NQL; ++ql)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf)
                    cd[it][ql][hf] = ldg_stream_v4(tb + (it * 16 + hf * 8 + g) * CPT + ql * 64 + c * 16);
        uint32_t scw[4][2][NG / 4];
#pragma unroll
        for (int it = 0; it < 4; ++it)
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const uint32_t* sp = reinterpret_cast<const uint32_t*>(tb + 64 * CPT + (it * 16 + hf * 8 + g) * NG);
#pragma unroll
                for (int i = 0; i < NG / 4; ++i) scw[it][hf][i] = __ldg(sp + i);
            }

        float m = -INFINITY;
#pragma unroll
        for (int it = 0; it < 4; ++it) {
            float srow[2] = {0.f, 0.f};
#pragma unroll
            for (int ql = 0; ql < NQL; ++ql) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
                const uint32_t wa[4] = {cd[it][ql][0].x, cd[it][ql][0].y, cd[it][ql][0].z, cd[it][ql][0].w};
                const uint32_t wb[4] = {cd[it][ql][1].x, cd[it][ql][1].y, cd[it][ql][1].z, cd[it][ql][1].w};
#pragma unroll
                for (int wd = 0; wd < 4; ++wd) {
                    uint32_t pa[4], pb[4];
                    unpack8<FMT>(wa[wd], pa);
                    unpack8<FMT>(wb[wd], pb);
                    mma_f16_16816(acc, pa[0], pb[0], pa[1], pb[1], qf[ql][4 * wd + 0], qf[ql][4 * wd + 1]);
                    mma_f16_16816(acc, pa[2], pb[2], pa[3], pb[3], qf[ql][4 * wd + 2], qf[ql][4 * wd + 3]);
                }
                // acc[0], acc[1]: row g, columns 2c, 2c+1; acc[2], acc[3]: row g + 8.  (lanes c >= 2: zeros)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int gi = 4 * ql + 2 * (c & 1);               // first of this lane's two groups
                    const uint32_t sw = scw[it][hf][ql];               // scale bytes of groups 4ql .. 4ql+3
                    float s0 = scale_to_f32<FMT>((sw >> (8 * (gi & 3))) & 0xffu);
                    float s1 = scale_to_f32<FMT>((sw >> (8 * ((gi & 3) + 1))) & 0xffu);
                    float d = fmaf(acc[2 * hf], s0, acc[2 * hf + 1] * s1);
                    if (GPH == 4) d += __shfl_xor_sync(0xffffffffu, d, 1);   // the head's other two groups
                    d *= ps[ql];
                    float contrib = wq[ql] * fmaxf(d, 0.f);
                    if (GPH == 4 && (c & 1)) contrib = 0.f;           // counted once
                    srow[hf] += contrib;
                }
            }
            // heads are split over quad lanes 0 and 1
            float sa = srow[0] + __shfl_xor_sync(0xffffffffu, srow[0], 1);
            float sb = srow[1] + __shfl_xor_sync(0xffffffffu, srow[1], 1);
            const int ta = t0 + it * 16 + g, tbk = ta + 8;
            if (ta < L) m = fmaxf(m, sa);
            if (tbk < L) m = fmaxf(m, sb);
        }
        if (c != 0) m = -INFINITY;
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 4));
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 8));
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 16));
        if (lane == 0) scores[(int64_t)b * nb_stride + tile] = m;
    }
}

template <int H, int D_IDX>
spot_status launch_score(const spot_select_params* p, float* scores, int nb_stride, cudaStream_t s) {
    // every warp gets the same number of 64-token tiles: with T tiles per sequence and room for `cap_warps` warps
    // per sequence (4 CTAs per SM in all), tiles per warp = ceil(T / cap_warps) and just enough warps for that.
    // (A grid-stride loop over a fixed 4 CTAs/SM grid left 3.46 tiles per warp at L = 128K, B = 4: a quarter of the
    // warps ran a 4th tile while the others idled -- profiles/r1_decode_cfg3_launches.md.)
    const int n_b_max = (p->max_seq_len + 63) / 64;
    const int cap_warps = max(1, (sm_count() * 4 * SCORE_WARPS) / p->B);
    const int tiles_per_warp = (n_b_max + cap_warps - 1) / cap_warps;
    const int warps = (n_b_max + tiles_per_warp - 1) / tiles_per_warp;
    dim3 grid((unsigned)((warps + SCORE_WARPS - 1) / SCORE_WARPS), (unsigned)p->B);
    const dim3 block(SCORE_WARPS * 32);
    if (p->fmt == SPOT_SELK_BF16) {
        SPOT_CUDA_TRY(launch_pdl(score_decode_bf16_kernel<H, D_IDX>, grid, block, 0, s, p->sel_q, p->w,
                                 (const uint16_t*)p->sel_k, p->cache_stride_tokens, p->seq_len, scores, nb_stride));
    } else if (p->fmt == SPOT_SELK_MXFP4) {
        SPOT_CUDA_TRY(launch_pdl(score_decode_q4_kernel<H, D_IDX, SPOT_SELK_MXFP4>, grid, block, 0, s, p->sel_q, p->w,
                                 (const uint8_t*)p->sel_k, p->cache_stride_tokens / 64, p->seq_len, scores, nb_stride));
    } else {
        SPOT_CUDA_TRY(launch_pdl(score_decode_q4_kernel<H, D_IDX, SPOT_SELK_INT4_E4M3>, grid, block, 0, s, p->sel_q,
                                 p->w, (const uint8_t*)p->sel_k, p->cache_stride_tokens / 64, p->seq_len, scores,
                                 nb_stride));
    }
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}

}  // namespace

// scores: fp32 [B][nb_stride]
spot_status score_decode(const spot_select_params* p, float* scores, int nb_stride, cudaStream_t s) {
    if (p->H_idx == 4 && p->d_idx == 64) return launch_score<4, 64>(p, scores, nb_stride, s);
    if (p->H_idx == 4 && p->d_idx == 128) return launch_score<4, 128>(p, scores, nb_stride, s);
    return SPOT_ERR_UNSUPPORTED;
}

}  // namespace spot
