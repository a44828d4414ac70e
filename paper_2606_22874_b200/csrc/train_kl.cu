// f4 -- the training-side reductions of one sequence (readings R34-R36):
//   teacher  p^tau[q,t]   = (1/H_q) sum_h softmax_t(sm_scale q_h . k_{g(h),t})      (Eq. 1: softmax, THEN mean over heads)
//   student  p^sigma[q,t] = softmax_t(s_s[q,t]),  s_s = sum_h w_h ReLU(q^I_h . k^I_{h,t})          (Eq. 2)
//   DenseKL[q]  = sum_{t<=q} p^tau log(p^tau / p^sigma)                                                        (Eq. 3)
//   SparseKL[q] = the same over S_q, both distributions renormalised there                                    (Eq. 4)
// with S_q the tokens of the top_k best blocks of query q by block-max score (Eq. 6 applied per query, R35).
//
// No L x L matrix is ever stored.  Two passes over the causal (query, key) plane, the selection kernel in between:
//   pass 1  per (query, head) the log-sum-exp of the teacher logits; per query the log-sum-exp of the student scores and
//           its block maxima s_bar[q, b]                                          -> workspace
//   select  select_hist_kernel in its decode form on L rows (row q sees q + 1 tokens), top-K -> block lists -> bit masks
//   pass 2  per (query, key): p^tau from the stored log-sum-exps (a sum over ALL heads: the one cross-warp step), the
//           student log-probability, membership of the key's block in S_q; per query the four running sums the two KLs
//           are made of.
// A CTA owns 32 / G queries (G = H_q / H_kv) and walks its visible keys in tiles of 32.  Warps 0-7: one KV head each,
// rows of the MMA = (query, head of the group), query-major, so that the head sum of Eq. 1 is a shuffle over row lanes;
// warp 8: the selector scores of the same tile.  Every warp streams its own operand through a private cp.async ring (as
// in attn_decode.cu); mma.sync m16n8k16, fp32 accumulate.
// Pass 1 on the tensor cores (round 2): when L is whole 64-query blocks the teacher's log-sum-exps come from the prefill
// attention kernel in its statistics-only form (attn_prefill_tc.cu, tcgen05 / TMEM / TMA) and the student's part from
// score_prefill_kernel in its rows form (score_prefill.cu: per query the block maxima and a log-sum-exp in 64-key pieces, folded
// by student_combine_rows_kernel) -- or, for selectors of fewer than four heads, from student_pass1_kernel below (mma.sync);
// train_pass_kernel<1> then serves ragged L only.  Pass 2 runs on
// train_pass2_tc_kernel (tcgen05) for the same whole-block sequences, on train_pass_kernel<2> otherwise.
#include "select_common.cuh"
#include "tc100.cuh"

#include <string.h>

namespace spot {

spot_status run_select(const spot_select_params* p, const float* scores, int nb_stride, int rows_per_seq, int max_nb,
                       const StepSync* sync, cudaStream_t s);                                   // select.cu
spot_status attn_prefill_stats(const uint16_t* q, const uint16_t* k, int64_t k_stride_token, int64_t k_stride_head, int L,
                               int H_q, int H_kv, float sm_scale, float* lse2, cudaStream_t stream);   // attn_prefill_tc.cu

spot_status score_prefill_rows(const uint16_t* sel_q, const float* w, const uint16_t* sel_k, int L, int H_idx, int d_idx,
                               int blk, float* blk_scores, int stride, float2* part, cudaStream_t s);   // score_prefill.cu

namespace {

constexpr int TR_KT = 32;                       // keys per tile
constexpr int TR_TW = 8;                        // teacher warps = KV heads per CTA
constexpr int TR_THREADS = (TR_TW + 1) * 32;
constexpr int TR_STAGES = 2;
constexpr int TR_D = 128;
constexpr int TR_KSTAGE = TR_KT * TR_D * 2;     // 8 KiB: one K sub-tile of one KV head
constexpr int TR_QMAX = 16;                     // queries per CTA at most (G = 2)

struct TrainArgs {
    const uint16_t* q;           // [L][H_q][128]
    const uint16_t* k;           // token / head strides in elements
    int64_t k_st, k_sh;
    const uint16_t* sel_q;       // [L][H][d]
    const float* w;              // [L][H]
    const uint16_t* sel_k;       // [L][H][d]
    int L, H_q, H_kv, G, H_idx, d_idx, blk;
    float scale_log2;
    float* t_lse2;               // [L][H_q] log2-domain log-sum-exp of the scaled teacher logits
    float* s_lse;                // [L] natural-log log-sum-exp of the student scores
    float* sp_part;              // [L][sp_nch][2]: (max, sum) of a query's student scores over one chunk of keys (student_pass1_kernel)
    int sp_nch;                  // chunks of SP_CHUNK key tiles per row
    float* p2_part;              // [chunks][L][4]: per-chunk sums of train_pass2_tc_kernel (P2_KT_CHUNK key tiles per chunk)
    float* blk_scores;           // [L][nb_stride]
    int nb_stride;
    const uint32_t* mask;        // [L][mask_stride] bit b: block b is in S_q
    int mask_stride;
    float* dense_kl;
    float* sparse_kl;
    float* teacher_lse;          // optional, natural log
};

__device__ __forceinline__ uint32_t tr_sw(int row, int chunk, int row_bytes) {
    return (uint32_t)(row * row_bytes + ((chunk ^ (row & 7)) << 4));
}

// rows x row_bytes from global (row stride in elements) into a swizzled stage; rows at or past n_valid are zero-filled
__device__ __forceinline__ void tr_issue(uint32_t stage, const uint16_t* base, int64_t stride, int row0, int n_rows_total,
                                         int row_bytes, int lane) {
    const int chunks = row_bytes >> 4;
    for (int id = lane; id < TR_KT * chunks; id += 32) {
        const int row = id / chunks, ch = id - row * chunks;
        const bool ok = row0 + row < n_rows_total;
        cp_async16(stage + tr_sw(row, ch, row_bytes), base + (int64_t)(ok ? row0 + row : 0) * stride + ch * 8, ok);
    }
}

template <int PASS>
__global__ void __launch_bounds__(TR_THREADS, 1) train_pass_kernel(TrainArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, c = lane & 3;
    const int G = a.G, QPT = 16 / G, QPC = 2 * QPT;
    const int n_tiles_q = (a.L + QPC - 1) / QPC;
    const int q0 = (n_tiles_q - 1 - (int)blockIdx.x) * QPC;            // heaviest (latest) queries first
    const int q_end = min(q0 + QPC, a.L);                              // one past the CTA's last query
    const int n_kt = (q_end + TR_KT - 1) / TR_KT;                      // key tiles: keys 0 .. q_end - 1
    const int srow_bytes = a.H_idx * a.d_idx * 2;                      // one token of the selector cache
    // shared memory: [8 warps][2 stages][8 KiB] K | [2 stages][32 x srow_bytes] selector K | sP[2][16][32] | sS[2][16][32]
    const uint32_t k_ring = smem_u32(smem) + warp * (TR_STAGES * TR_KSTAGE);
    const uint32_t s_ring = smem_u32(smem) + TR_TW * TR_STAGES * TR_KSTAGE;
    float* sP = reinterpret_cast<float*>(smem + TR_TW * TR_STAGES * TR_KSTAGE + TR_STAGES * TR_KT * srow_bytes);
    float* sS = sP + 2 * TR_QMAX * TR_KT;
    const uint32_t sQ = smem_u32(sS + 2 * TR_QMAX * TR_KT);            // student: its 16 query rows, swizzled like a key tile
    if (PASS == 2) {
        for (int e = threadIdx.x; e < 2 * TR_QMAX * TR_KT; e += TR_THREADS) sP[e] = 0.f;
        __syncthreads();
    }

    // ------------------------------------------------------------------------------------------------------------
    // per-warp state
    // ------------------------------------------------------------------------------------------------------------
    const bool teacher = warp < TR_TW && warp < a.H_kv;
    const bool student = warp == TR_TW;
    uint32_t qf[2][8][4];                       // teacher: Q fragments of the two m-tiles
    float swt[4][2];                            // student: w_h of rows g and g + 8
    float st_m[2][2], st_l[2][2];               // pass 1: online (max, sum) of rows (m-tile j, half)
    float row_lse[2][2];                        // pass 2 (teacher): log2-domain LSE of the rows
    float bm[2] = {-INFINITY, -INFINITY};       // pass 1 (student): running maximum of the current key block
    const int ks_sel = a.d_idx >> 4;            // k-steps per selector head
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) { st_m[j][hf] = -INFINITY; st_l[j][hf] = 0.f; row_lse[j][hf] = 0.f; }

    // row r of m-tile j: query q0 + j QPT + r / G, head hk G + r % G (query-major: the heads of a query sit on
    // consecutive row lanes)
    auto row_query = [&](int j, int r) -> int { return q0 + j * QPT + r / G; };
    if (teacher) {
        const int hk = warp;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int ra = g, rb = g + 8;
            const int qa = row_query(j, ra), qb = row_query(j, rb);
            const uint16_t* pa = a.q + ((int64_t)qa * a.H_q + hk * G + ra % G) * TR_D;
            const uint16_t* pb = a.q + ((int64_t)qb * a.H_q + hk * G + rb % G) * TR_D;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                const int col = ks * 16 + c * 2;
                qf[j][ks][0] = qa < a.L ? *reinterpret_cast<const uint32_t*>(pa + col) : 0u;
                qf[j][ks][1] = qb < a.L ? *reinterpret_cast<const uint32_t*>(pb + col) : 0u;
                qf[j][ks][2] = qa < a.L ? *reinterpret_cast<const uint32_t*>(pa + col + 8) : 0u;
                qf[j][ks][3] = qb < a.L ? *reinterpret_cast<const uint32_t*>(pb + col + 8) : 0u;
            }
            if (PASS == 2) {
                row_lse[j][0] = qa < a.L ? a.t_lse2[(int64_t)qa * a.H_q + hk * G + ra % G] : 0.f;
                row_lse[j][1] = qb < a.L ? a.t_lse2[(int64_t)qb * a.H_q + hk * G + rb % G] : 0.f;
            }
        }
    }
    if (student) {
        // rows = the CTA's queries (QPC <= 16), the rest zero
        const int qa = q0 + g, qb = q0 + g + 8;
        const bool va = g < QPC && qa < a.L, vb = g + 8 < QPC && qb < a.L;
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            swt[h][0] = (va && h < a.H_idx) ? a.w[(int64_t)qa * a.H_idx + h] : 0.f;
            swt[h][1] = (vb && h < a.H_idx) ? a.w[(int64_t)qb * a.H_idx + h] : 0.f;
        }
        // the selector queries go to shared memory once (their fragments would cost 128 registers at d_idx = 128)
        const int chunks = srow_bytes >> 4;
        for (int id = lane; id < 16 * chunks; id += 32) {
            const int row = id / chunks, ch = id - row * chunks;
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (row < QPC && q0 + row < a.L)
                v = *reinterpret_cast<const uint4*>(a.sel_q + (int64_t)(q0 + row) * (a.H_idx * a.d_idx) + ch * 8);
            asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(sQ + tr_sw(row, ch, srow_bytes)), "r"(v.x), "r"(v.y),
                         "r"(v.z), "r"(v.w) : "memory");
        }
        __syncwarp();
    }

    // pass 2: the KL sums of this thread's (query, key lane) elements: element e = tid + 256 i -> query e / 32, lane e % 32
    float acc_d[2] = {0.f, 0.f}, acc_a[2] = {0.f, 0.f}, acc_b[2] = {0.f, 0.f}, acc_c[2] = {0.f, 0.f};
    float my_slse[2] = {0.f, 0.f};
    if (PASS == 2 && warp < TR_TW) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int q = q0 + warp + 8 * i;
            if (warp + 8 * i < QPC && q < a.L) my_slse[i] = a.s_lse[q];
        }
    }

    // ------------------------------------------------------------------------------------------------------------
    // the key loop
    // ------------------------------------------------------------------------------------------------------------
    auto issue = [&](int kt) {
        if (teacher) tr_issue(k_ring + (kt % TR_STAGES) * TR_KSTAGE, a.k + (int64_t)warp * a.k_sh, a.k_st, kt * TR_KT, q_end,
                              TR_D * 2, lane);
        if (student) tr_issue(s_ring + (kt % TR_STAGES) * (TR_KT * srow_bytes), a.sel_k, a.H_idx * a.d_idx, kt * TR_KT, q_end,
                              srow_bytes, lane);
        cp_async_commit();
    };
    issue(0);
    for (int kt = 0; kt < n_kt; ++kt) {
        if (kt + 1 < n_kt) issue(kt + 1); else cp_async_commit();
        cp_async_wait<1>();
        __syncwarp();
        const int t0 = kt * TR_KT, buf = kt & 1;
        const int mi = lane >> 3, r8 = lane & 7;

        if (teacher) {
            const uint32_t kb = k_ring + (kt % TR_STAGES) * TR_KSTAGE;
            float s[2][4][4];
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) s[j][nt][0] = s[j][nt][1] = s[j][nt][2] = s[j][nt][3] = 0.f;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    uint32_t b0, b1, b2, b3;
                    ldmatrix_x4(b0, b1, b2, b3, kb + tr_sw(half * 16 + (mi >> 1) * 8 + r8, 2 * ks + (mi & 1), TR_D * 2));
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        mma_bf16_16816(s[j][half * 2], qf[j][ks][0], qf[j][ks][1], qf[j][ks][2], qf[j][ks][3], b0, b1);
                        mma_bf16_16816(s[j][half * 2 + 1], qf[j][ks][0], qf[j][ks][1], qf[j][ks][2], qf[j][ks][3], b2, b3);
                    }
                }
            // log2 domain, causal mask (key <= query) and rows past the sequence
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int q = row_query(j, g + 8 * hf);
                    float v[8];
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int key = t0 + nt * 8 + c * 2 + e;
                            v[nt * 2 + e] = (q < a.L && key <= q) ? s[j][nt][hf * 2 + e] * a.scale_log2 : -INFINITY;
                        }
                    if (PASS == 1) {
                        float mx = v[0];
#pragma unroll
                        for (int i = 1; i < 8; ++i) mx = fmaxf(mx, v[i]);
                        const float mn = fmaxf(st_m[j][hf], mx);
                        if (mn > -INFINITY) {
                            float sum = 0.f;
#pragma unroll
                            for (int i = 0; i < 8; ++i) sum += fast_exp2(v[i] - mn);
                            st_l[j][hf] = st_l[j][hf] * fast_exp2(st_m[j][hf] - mn) + sum;
                            st_m[j][hf] = mn;
                        }
                    } else {
                        // p_h = exp2(v - lse_h); Eq. 1's sum over the heads of the group = over the G row lanes of the query
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            float p = fast_exp2(v[i] - row_lse[j][hf]);
                            if (G >= 2) p += __shfl_xor_sync(0xffffffffu, p, 4);
                            if (G >= 4) p += __shfl_xor_sync(0xffffffffu, p, 8);
                            if (G >= 8) p += __shfl_xor_sync(0xffffffffu, p, 16);
                            v[i] = p;
                        }
                        // (G == 16: rows g and g + 8 are the same query -- both halves add into its slot)
                        const int r = g + 8 * hf;
                        if (r % G == 0 || (G == 16 && g == 0)) {
                            const int ql = j * QPT + r / G;
#pragma unroll
                            for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                                for (int e = 0; e < 2; ++e)
                                    atomicAdd(&sP[(buf * TR_QMAX + ql) * TR_KT + nt * 8 + c * 2 + e], v[nt * 2 + e]);
                        }
                    }
                }
        }

        if (student) {
            const uint32_t sb = s_ring + (kt % TR_STAGES) * (TR_KT * srow_bytes);
            float sv[4][4];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) sv[nt][0] = sv[nt][1] = sv[nt][2] = sv[nt][3] = 0.f;
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                if (h < a.H_idx) {
                    float acc[4][4];
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        if (ks < ks_sel) {
                            const int ch0 = h * (a.d_idx >> 3) + 2 * ks;
                            uint32_t a0, a1, a2, a3;
                            ldmatrix_x4(a0, a1, a2, a3, sQ + tr_sw((mi & 1) * 8 + r8, ch0 + (mi >> 1), srow_bytes));
#pragma unroll
                            for (int half = 0; half < 2; ++half) {
                                uint32_t b0, b1, b2, b3;
                                ldmatrix_x4(b0, b1, b2, b3, sb + tr_sw(half * 16 + (mi >> 1) * 8 + r8, ch0 + (mi & 1), srow_bytes));
                                mma_bf16_16816(acc[half * 2], a0, a1, a2, a3, b0, b1);
                                mma_bf16_16816(acc[half * 2 + 1], a0, a1, a2, a3, b2, b3);
                            }
                        }
                    }
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        sv[nt][0] = fmaf(swt[h][0], fmaxf(acc[nt][0], 0.f), sv[nt][0]);
                        sv[nt][1] = fmaf(swt[h][0], fmaxf(acc[nt][1], 0.f), sv[nt][1]);
                        sv[nt][2] = fmaf(swt[h][1], fmaxf(acc[nt][2], 0.f), sv[nt][2]);
                        sv[nt][3] = fmaf(swt[h][1], fmaxf(acc[nt][3], 0.f), sv[nt][3]);
                    }
                }
            }
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const int ql = g + 8 * hf, q = q0 + ql;
                const bool rowok = ql < QPC && q < a.L;
                if (PASS == 1) {
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        const int key0 = t0 + nt * 8;
                        float v0 = (rowok && key0 + c * 2 <= q) ? sv[nt][hf * 2] : -INFINITY;
                        float v1 = (rowok && key0 + c * 2 + 1 <= q) ? sv[nt][hf * 2 + 1] : -INFINITY;
                        // online log-sum-exp of the row (natural log; this thread's columns, merged over the quad at the end)
                        const float mx = fmaxf(v0, v1), mn = fmaxf(st_m[0][hf], mx);
                        if (mn > -INFINITY) {
                            st_l[0][hf] = st_l[0][hf] * __expf(st_m[0][hf] - mn) + __expf(v0 - mn) + __expf(v1 - mn);
                            st_m[0][hf] = mn;
                        }
                        // block maxima: flushed when the 8 keys end a block
                        bm[hf] = fmaxf(bm[hf], mx);
                        if ((key0 + 8) % a.blk == 0 || (kt == n_kt - 1 && nt == 3)) {
                            float m = bm[hf];
                            m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));
                            m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
                            if (c == 0 && m > -INFINITY) a.blk_scores[(int64_t)q * a.nb_stride + key0 / a.blk] = m;
                            bm[hf] = -INFINITY;
                        }
                    }
                } else if (ql < TR_QMAX) {
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        sS[(buf * TR_QMAX + ql) * TR_KT + nt * 8 + c * 2] = sv[nt][hf * 2];
                        sS[(buf * TR_QMAX + ql) * TR_KT + nt * 8 + c * 2 + 1] = sv[nt][hf * 2 + 1];
                    }
                }
            }
        }

        if (PASS == 2) {
            __syncthreads();                    // the tile's head sums and student scores are in shared memory
            if (warp < TR_TW) {
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int ql = warp + 8 * i, q = q0 + ql, t = t0 + lane;
                    if (ql < QPC) {
                        const int at = (buf * TR_QMAX + ql) * TR_KT + lane;
                        const float pt = sP[at] / (float)a.H_q;
                        sP[at] = 0.f;                                   // re-armed for tile kt + 2
                        if (q < a.L && t <= q) {
                            const float lps = sS[at] - my_slse[i];      // log p^sigma
                            const int b = t / a.blk;
                            const bool in_s = (a.mask[(int64_t)q * a.mask_stride + (b >> 5)] >> (b & 31)) & 1u;
                            if (in_s) acc_b[i] += __expf(lps);
                            if (pt > 0.f) {
                                const float term = pt * (__logf(pt) - lps);
                                acc_d[i] += term;
                                if (in_s) { acc_a[i] += pt; acc_c[i] += term; }
                            }
                        }
                    }
                }
            }
        }
        __syncwarp();                           // the stage is free for the request after next
    }
    cp_async_wait<0>();

    // ------------------------------------------------------------------------------------------------------------
    // results
    // ------------------------------------------------------------------------------------------------------------
    if (PASS == 1) {
        if (teacher) {
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    float m = st_m[j][hf], l = st_l[j][hf];
#pragma unroll
                    for (int o = 1; o <= 2; o <<= 1) {
                        const float m2 = __shfl_xor_sync(0xffffffffu, m, o), l2 = __shfl_xor_sync(0xffffffffu, l, o);
                        const float M = fmaxf(m, m2);
                        if (M > -INFINITY) { l = l * fast_exp2(m - M) + l2 * fast_exp2(m2 - M); m = M; }
                    }
                    const int r = g + 8 * hf, q = row_query(j, r);
                    if (c == 0 && q < a.L) {
                        const float lse2 = m + log2f(l);
                        a.t_lse2[(int64_t)q * a.H_q + warp * G + r % G] = lse2;
                        if (a.teacher_lse) a.teacher_lse[(int64_t)q * a.H_q + warp * G + r % G] = lse2 * 0.6931471805599453f;
                    }
                }
        }
        if (student) {
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                float m = st_m[0][hf], l = st_l[0][hf];
#pragma unroll
                for (int o = 1; o <= 2; o <<= 1) {
                    const float m2 = __shfl_xor_sync(0xffffffffu, m, o), l2 = __shfl_xor_sync(0xffffffffu, l, o);
                    const float M = fmaxf(m, m2);
                    if (M > -INFINITY) { l = l * __expf(m - M) + l2 * __expf(m2 - M); m = M; }
                }
                const int ql = g + 8 * hf, q = q0 + ql;
                if (c == 0 && ql < QPC && q < a.L) a.s_lse[q] = m + __logf(l);
            }
        }
    } else if (warp < TR_TW) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            float d = acc_d[i], A = acc_a[i], B = acc_b[i], C = acc_c[i];
#pragma unroll
            for (int o = 16; o; o >>= 1) {
                d += __shfl_xor_sync(0xffffffffu, d, o);
                A += __shfl_xor_sync(0xffffffffu, A, o);
                B += __shfl_xor_sync(0xffffffffu, B, o);
                C += __shfl_xor_sync(0xffffffffu, C, o);
            }
            const int ql = warp + 8 * i, q = q0 + ql;
            if (lane == 0 && ql < QPC && q < a.L) {
                a.dense_kl[q] = d;
                // Eq. 4: sum_S (p/A) log((p/A) / (s/B)) = C / A - log A + log B
                a.sparse_kl[q] = A > 0.f ? C / A - __logf(A) + __logf(B) : 0.f;
            }
        }
    }
}

// ---- pass 1, the student's part alone (used when the teacher's statistics come from the tcgen05 kernel) -------------------
// s_lse[q] = log sum_{t <= q} exp(s_s[q, t]) and the block maxima s_bar[q, b] of every query.  A CTA owns 64 consecutive queries,
// one m16 tile per warp, and walks the visible keys in tiles of 64 that all four warps share: the selector key rows are loaded
// once per CTA (cooperative cp.async ring) and used by 64 queries -- in train_pass_kernel<1> a single warp per CTA served 8
// queries through a ring of its own and the pass took as long as the teacher's (19.5 ms of 21.6 at L = 16K).
// (round 2, later) The causal triangle is cut along the keys too: CTA (chunk c, query tile) walks 32 key tiles of 32 keys only
// and leaves one (max, sum) pair per query, which student_combine_kernel folds into s_lse.  One CTA per 64 queries over the whole
// row had 256 CTAs of four warps for 148 SMs, the heaviest one alone on the critical path (1.9 ms at L = 16K, tensor pipe 6 %,
// 26 % issue utilisation with one or two warps per scheduler); 1024-key chunks of 32-key tiles (64 KiB of shared memory: three
// CTAs per SM) bring spot_train_kl at L = 16K from 5.80 to 4.72 ms.
constexpr int SP_WARPS = 4;
constexpr int SP_THREADS = SP_WARPS * 32;
constexpr int SP_QPC = SP_WARPS * 16;
constexpr int SP_KT = 32;
constexpr int SP_CHUNK = 32;                   // key tiles per CTA (1024 keys)

__global__ void __launch_bounds__(SP_THREADS) student_pass1_kernel(TrainArgs a, int stages) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, c = lane & 3, mi = lane >> 3, r8 = lane & 7;
    const int n_tiles_q = (a.L + SP_QPC - 1) / SP_QPC;
    const int q0 = (n_tiles_q - 1 - (int)blockIdx.y) * SP_QPC;         // heaviest (latest) queries first
    const int q_end = min(q0 + SP_QPC, a.L);
    const int kt_lo = (int)blockIdx.x * SP_CHUNK;
    const int n_kt = min((q_end + SP_KT - 1) / SP_KT, kt_lo + SP_CHUNK);   // this CTA's key tiles: [kt_lo, n_kt)
    if (kt_lo >= n_kt) return;                                          // the chunk lies past the tile's diagonal
    const int srow_bytes = a.H_idx * a.d_idx * 2;
    const int chunks = srow_bytes >> 4;
    const int stage_bytes = SP_KT * srow_bytes;
    const uint32_t ring = smem_u32(smem);
    const uint32_t sQ = ring + stages * stage_bytes + warp * 16 * srow_bytes;   // this warp's 16 query rows
    const int ks_sel = a.d_idx >> 4;
    const int qw0 = q0 + warp * 16;                                     // the warp's first query
    const int qa = qw0 + g, qb = qw0 + g + 8;
    const bool va = qa < a.L, vb = qb < a.L;
    float swt[4][2];
#pragma unroll
    for (int h = 0; h < 4; ++h) {
        swt[h][0] = (va && h < a.H_idx) ? a.w[(int64_t)qa * a.H_idx + h] : 0.f;
        swt[h][1] = (vb && h < a.H_idx) ? a.w[(int64_t)qb * a.H_idx + h] : 0.f;
    }
    for (int id = lane; id < 16 * chunks; id += 32) {
        const int row = id / chunks, ch = id - row * chunks;
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (qw0 + row < a.L) v = *reinterpret_cast<const uint4*>(a.sel_q + (int64_t)(qw0 + row) * (a.H_idx * a.d_idx) + ch * 8);
        asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(sQ + tr_sw(row, ch, srow_bytes)), "r"(v.x), "r"(v.y),
                     "r"(v.z), "r"(v.w) : "memory");
    }
    __syncwarp();
    float st_m[2] = {-INFINITY, -INFINITY}, st_l[2] = {0.f, 0.f}, bm[2] = {-INFINITY, -INFINITY};

    const int csh = (chunks & (chunks - 1)) == 0 ? 31 - __clz(chunks) : -1;    // 16-byte chunks per row: a power of two as a rule
    auto issue = [&](int kt) {
        if (kt < n_kt) {
            const uint32_t stage = ring + (kt % stages) * stage_bytes;
            for (int id = tid; id < SP_KT * chunks; id += SP_THREADS) {
                const int row = csh >= 0 ? id >> csh : id / chunks, ch = id - row * chunks;
                const bool ok = kt * SP_KT + row < q_end;
                cp_async16(stage + tr_sw(row, ch, srow_bytes),
                           a.sel_k + (int64_t)(ok ? kt * SP_KT + row : 0) * (a.H_idx * a.d_idx) + ch * 8, ok);
            }
        }
        cp_async_commit();
    };
    for (int i = 0; i < stages - 1; ++i) issue(kt_lo + i);
    for (int kt = kt_lo; kt < n_kt; ++kt) {
        issue(kt + stages - 1);                 // (into the stage every warp left at the end of iteration kt - 1)
        if (stages == 3) cp_async_wait<2>(); else cp_async_wait<1>();
        __syncthreads();                        // tile kt has landed for every thread
        const uint32_t stage = ring + (kt % stages) * stage_bytes;
        // the warp's last query is qw0 + 15: tiles past it hold no visible key for this warp
        if (kt * SP_KT <= min(qw0 + 15, a.L - 1)) {
#pragma unroll 1
            for (int sub = 0; sub < SP_KT / 32; ++sub) {
                const int t0 = kt * SP_KT + sub * 32;
                if (t0 > min(qw0 + 15, a.L - 1)) break;
                const uint32_t sb = stage + sub * 32 * srow_bytes;
                float sv[4][4];
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) sv[nt][0] = sv[nt][1] = sv[nt][2] = sv[nt][3] = 0.f;
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    if (h < a.H_idx) {
                        float acc[4][4];
#pragma unroll
                        for (int nt = 0; nt < 4; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks) {
                            if (ks < ks_sel) {
                                const int ch0 = h * (a.d_idx >> 3) + 2 * ks;
                                uint32_t a0, a1, a2, a3;
                                ldmatrix_x4(a0, a1, a2, a3, sQ + tr_sw((mi & 1) * 8 + r8, ch0 + (mi >> 1), srow_bytes));
#pragma unroll
                                for (int half = 0; half < 2; ++half) {
                                    uint32_t b0, b1, b2, b3;
                                    ldmatrix_x4(b0, b1, b2, b3,
                                                sb + tr_sw(half * 16 + (mi >> 1) * 8 + r8, ch0 + (mi & 1), srow_bytes));
                                    mma_bf16_16816(acc[half * 2], a0, a1, a2, a3, b0, b1);
                                    mma_bf16_16816(acc[half * 2 + 1], a0, a1, a2, a3, b2, b3);
                                }
                            }
                        }
#pragma unroll
                        for (int nt = 0; nt < 4; ++nt) {
                            sv[nt][0] = fmaf(swt[h][0], fmaxf(acc[nt][0], 0.f), sv[nt][0]);
                            sv[nt][1] = fmaf(swt[h][0], fmaxf(acc[nt][1], 0.f), sv[nt][1]);
                            sv[nt][2] = fmaf(swt[h][1], fmaxf(acc[nt][2], 0.f), sv[nt][2]);
                            sv[nt][3] = fmaf(swt[h][1], fmaxf(acc[nt][3], 0.f), sv[nt][3]);
                        }
                    }
                }
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int q = qw0 + g + 8 * hf;
                    const bool rowok = q < a.L;
                    // the row's last key tile: its open block is flushed there (keys past q are masked)
                    const bool last_sub = t0 + 32 > q;
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        const int key0 = t0 + nt * 8;
                        float v0 = (rowok && key0 + c * 2 <= q) ? sv[nt][hf * 2] : -INFINITY;
                        float v1 = (rowok && key0 + c * 2 + 1 <= q) ? sv[nt][hf * 2 + 1] : -INFINITY;
                        const float mx = fmaxf(v0, v1), mn = fmaxf(st_m[hf], mx);
                        if (mn > -INFINITY) {
                            st_l[hf] = st_l[hf] * __expf(st_m[hf] - mn) + __expf(v0 - mn) + __expf(v1 - mn);
                            st_m[hf] = mn;
                        }
                        bm[hf] = fmaxf(bm[hf], mx);
                        if ((key0 + 8) % a.blk == 0 || (last_sub && nt == 3)) {
                            float m = bm[hf];
                            m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));
                            m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
                            if (c == 0 && m > -INFINITY) a.blk_scores[(int64_t)q * a.nb_stride + key0 / a.blk] = m;
                            bm[hf] = -INFINITY;
                        }
                    }
                }
            }
        }
        __syncthreads();                        // every warp has left the stage before the request after next refills it
    }
    cp_async_wait<0>();
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
        float m = st_m[hf], l = st_l[hf];
#pragma unroll
        for (int o = 1; o <= 2; o <<= 1) {
            const float m2 = __shfl_xor_sync(0xffffffffu, m, o), l2 = __shfl_xor_sync(0xffffffffu, l, o);
            const float M = fmaxf(m, m2);
            if (M > -INFINITY) { l = l * __expf(m - M) + l2 * __expf(m2 - M); m = M; }
        }
        const int q = qw0 + g + 8 * hf;
        if (c == 0 && q < a.L)
            *reinterpret_cast<float2*>(a.sp_part + ((int64_t)q * a.sp_nch + blockIdx.x) * 2) = make_float2(m, l);
    }
}

// s_lse[q] = log sum exp over the chunks of keys row q can see (chunk c covers SP_CHUNK * SP_KT = 1024 keys from 1024 c)
__global__ void __launch_bounds__(256) student_combine_kernel(const float* __restrict__ part, int nch, float* __restrict__ s_lse,
                                                              int L) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= L) return;
    const int n = q / (SP_CHUNK * SP_KT) + 1;                 // chunks that hold a key t <= q
    float m = -INFINITY, l = 0.f;
    for (int i = 0; i < n && i < nch; ++i) {
        const float2 p = *reinterpret_cast<const float2*>(part + ((int64_t)q * nch + i) * 2);
        const float M = fmaxf(m, p.x);
        if (M > -INFINITY) { l = l * __expf(m - M) + p.y * __expf(p.x - M); m = M; }
    }
    s_lse[q] = m + __logf(l);
}

// the same for the rows form of score_prefill_kernel: part[j][q] = (max, sum exp) of row q over the 64 keys of block j.
// Thread (q, u) folds blocks u, u + 8, ..; the eight threads of a row (consecutive lanes) then fold their pairs.
__global__ void __launch_bounds__(256) student_combine_rows_kernel(const float2* __restrict__ part, float* __restrict__ s_lse, int L) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int q = t >> 3, u = t & 7;
    float m = -INFINITY, l = 0.f;
    if (q < L)
        for (int j = u; j <= q / 64; j += 8) {
            const float2 p = part[(int64_t)j * L + q];
            const float M = fmaxf(m, p.x);
            l = l * __expf(m - M) + p.y * __expf(p.x - M);   // (p.x is finite: every visible block holds a visible key)
            m = M;
        }
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, m, o), l2 = __shfl_xor_sync(0xffffffffu, l, o);
        const float M = fmaxf(m, m2);
        if (M > -INFINITY) { l = l * __expf(m - M) + l2 * __expf(m2 - M); m = M; }
    }
    if (q < L && u == 0) s_lse[q] = m + __logf(l);
}

// sum over the 32 lanes of v[j] for every j, delivered to lane j (31 shuffles instead of 32 x 5): at each level a lane keeps
// the half of its elements that its own bit selects and adds the partner's copy of that half
__device__ __forceinline__ float warp_transpose_sum(float (&v)[32], int lane) {
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const bool up = (lane & off) != 0;
#pragma unroll
        for (int k = 0; k < off; ++k) {
            const float send = up ? v[k] : v[k + off];
            const float keep = up ? v[k + off] : v[k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
    }
    return v[0];
}

// ---- pass 2 on the tensor cores (tcgen05 / TMEM / TMA) ----------------------------------------------------------------------
// The element-level head sum of Eq. 1 decides the layout.  The products are computed TRANSPOSED: S^T = K Q^T, the 128 keys of a
// tile are the M rows (TMEM lanes, one key per epilogue thread) and the (head of the group, query) pairs of a 64-query block the
// N columns.  A thread then sees, for ITS key, the logits of every head and every query in its own registers: the sum over the
// 32 heads is plain register arithmetic, head step after head step, and only the four KL sums of a query (over keys) cross
// lanes -- 4 values per (query, 32 keys) through a transposing shuffle tree instead of 32 per (query, key).
//   step      = one accumulator: a KV head's (up to 4 query heads x 64 queries) columns, or the student's 4 selector heads
//   stage     = the two operands of a step in shared memory (96 KiB: [columns][128 d] + [128 keys][128 d]), TMA ring of 2
//   TMEM      = two accumulators of 256 columns
//   warp 0 TMA producer, warp 1 MMA issuer (converged, one elected lane), warp 2 TMEM allocation, warps 4-11 epilogue:
//   lane quarter = warp & 3, query half = (warp - 4) >> 2 (32 queries each, so the running head sum is 32 registers).
// One CTA per 64-query block; it walks the visible keys in tiles of 128.
constexpr int P2_THREADS = 12 * 32;
constexpr int P2_QB = 64;                        // queries per CTA
constexpr int P2_KT = 128;                       // keys per tile
constexpr uint32_t P2_A_BYTES = 128 * 256;       // K tile: [2 d-halves][128 keys][128 B]  (student: [4 planes][128 keys][128 B] = 64 KiB)
constexpr uint32_t P2_STAGE = 96 * 1024;         // the larger operand (64 KiB) first, the smaller (32 KiB) behind it:
constexpr uint32_t P2_BIG = 0, P2_SMALL = 64 * 1024;   // teacher: B = queries (big), A = keys; student: A = keys (big), B = queries
constexpr uint32_t P2_SMEM_MISC = 16 * 1024;     // lse2 [32 heads][64] (8 KiB), w [4][64], s_lse [64], tile bits [2][64], sums, barriers
constexpr uint32_t P2_OFF_W = 8192, P2_OFF_SLSE = 9216, P2_OFF_BITS = 9472, P2_OFF_SUM = 9984, P2_OFF_BARS = 14080,
                   P2_OFF_TMEM = 14144;
constexpr uint32_t P2_SMEM = 1024 + 2 * P2_STAGE + P2_SMEM_MISC;

struct Pass2Args {
    const float* t_lse2;         // [L][H_q] log2 domain
    const float* s_lse;          // [L]
    const float* w;              // [L][4]
    const uint32_t* mask;        // [L][mask_stride]
    int mask_stride;
    int L, H_q, G, d_idx, blk;
    int hps;                     // query heads per teacher step: min(G, 4)
    int t_steps, s_steps;        // teacher steps (H_q / hps), student steps (d_idx / 64)
    float scale_log2;
    float* dense_kl;
    float* sparse_kl;
    // the causal triangle is cut along the keys too: CTA (query block, chunk c) walks key tiles [c kt_chunk, (c + 1) kt_chunk)
    // and leaves its four sums per query in part[c][q][4]; pass2_finalize_kernel adds the chunks and forms the two KLs.  (One
    // CTA per query block over all its keys: 256 CTAs of 1 .. 128 tiles on 148 SMs, the heaviest alone at the end.)
    float* part;
    int kt_chunk;
};

__global__ void __launch_bounds__(P2_THREADS, 1) train_pass2_tc_kernel(const __grid_constant__ CUtensorMap tm_q,
                                                                       const __grid_constant__ CUtensorMap tm_k,
                                                                       const __grid_constant__ CUtensorMap tm_sq,
                                                                       const __grid_constant__ CUtensorMap tm_sk,
                                                                       const Pass2Args a) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* smem = smem_raw + (base - smem_u32(smem_raw));
    unsigned char* misc = smem + 2 * P2_STAGE;
    const uint32_t misc_u32 = base + 2 * P2_STAGE;
    float* s_lse2 = reinterpret_cast<float*>(misc);                    // [H_q <= 32][64]
    float* s_w = reinterpret_cast<float*>(misc + P2_OFF_W);            // [4][64]
    float* s_slse = reinterpret_cast<float*>(misc + P2_OFF_SLSE);      // [64]
    uint32_t* s_bits = reinterpret_cast<uint32_t*>(misc + P2_OFF_BITS);   // [2][64] mask bits of the tile's blocks
    float* s_sum = reinterpret_cast<float*>(misc + P2_OFF_SUM);        // [4 lane quarters][64 q][4 sums]
    const uint32_t bars = misc_u32 + P2_OFF_BARS;
    const uint32_t bar_full = bars;            // [2] stage landed
    const uint32_t bar_empty = bars + 16;      // [2] stage read by its MMAs
    const uint32_t bar_t_full = bars + 32;     // [2] accumulator complete
    const uint32_t bar_t_empty = bars + 48;    // [2] accumulator read by the 8 epilogue warps
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(misc + P2_OFF_TMEM);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_qb = a.L / P2_QB;
    const int i = n_qb - 1 - (int)blockIdx.x;                          // heaviest (latest) query block first
    const int q0 = i * P2_QB;
    const int n_kt = (q0 + P2_QB + P2_KT - 1) / P2_KT;                 // key tiles: keys 0 .. q0 + 63
    const int kt_lo = (int)blockIdx.y * a.kt_chunk, kt_hi = min(n_kt, kt_lo + a.kt_chunk);   // this CTA's chunk of them
    if (kt_lo >= n_kt) return;                                         // (the whole CTA: the chunk lies past the diagonal)
    const int n_steps = a.t_steps + a.s_steps;

    if (threadIdx.x == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
            mbar_init(bar_t_full + 8 * s, 1);
            mbar_init(bar_t_empty + 8 * s, 8);
        }
        mbar_fence_init();
        tma_prefetch_desc(&tm_q); tma_prefetch_desc(&tm_k); tma_prefetch_desc(&tm_sq); tma_prefetch_desc(&tm_sk);
    }
    if (warp == 2) tmem_alloc(misc_u32 + P2_OFF_TMEM, 512);
    // the block's per-query constants: lse2 as [head][query] (a step reads 32 consecutive queries of one head), w as [h][q]
    for (int e = threadIdx.x; e < a.H_q * P2_QB; e += P2_THREADS) {
        const int q = e / a.H_q, h = e - q * a.H_q;
        s_lse2[h * P2_QB + q] = a.t_lse2[(int64_t)(q0 + q) * a.H_q + h];
    }
    for (int e = threadIdx.x; e < 4 * P2_QB; e += P2_THREADS) {
        const int q = e >> 2, h = e & 3;
        s_w[h * P2_QB + q] = a.w[(int64_t)(q0 + q) * 4 + h];
    }
    for (int e = threadIdx.x; e < P2_QB; e += P2_THREADS) s_slse[e] = a.s_lse[q0 + e];
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tbase = *tmem_slot;

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            int n = 0;
            for (int kt = kt_lo; kt < kt_hi; ++kt)
                for (int st = 0; st < n_steps; ++st, ++n) {
                    const int s = n & 1;
                    mbar_wait(bar_empty + 8 * s, ((n >> 1) & 1) ^ 1);
                    const uint32_t sb = base + s * P2_STAGE;
                    if (st < a.t_steps) {
                        const int head0 = st * a.hps, hk = head0 / a.G;
                        mbar_arrive_expect_tx(bar_full + 8 * s, (uint32_t)a.hps * 64u * 256u + P2_A_BYTES);
                        // B: [d-half][hps heads][64 queries][128 B]
                        tma_load_5d(sb + P2_BIG, &tm_q, bar_full + 8 * s, 0, q0, head0, 0, 0);
                        // A: [d-half][128 keys][128 B]
                        tma_load_5d(sb + P2_SMALL, &tm_k, bar_full + 8 * s, 0, kt * P2_KT, 0, hk, 0);
                    } else {
                        // the student's planes (128 B = 64 selector dims of one token): step u holds planes 4u .. 4u + 3
                        const int pl0 = (st - a.t_steps) * 4;
                        mbar_arrive_expect_tx(bar_full + 8 * s, 4u * 64u * 128u + 4u * 128u * 128u);
                        tma_load_4d(sb + P2_SMALL, &tm_sq, bar_full + 8 * s, 0, q0, pl0, 0);          // [4 planes][64 q][128 B]
                        tma_load_4d(sb + P2_BIG, &tm_sk, bar_full + 8 * s, 0, kt * P2_KT, pl0, 0);  // [4 planes][128 keys][128 B]
                    }
                }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer (converged; one elected lane issues) ================================
        int n = 0;
        for (int kt = kt_lo; kt < kt_hi; ++kt)
            for (int st = 0; st < n_steps; ++st, ++n) {
                const int s = n & 1;
                mbar_wait(bar_full + 8 * s, (n >> 1) & 1);
                mbar_wait(bar_t_empty + 8 * s, ((n >> 1) & 1) ^ 1);    // (accumulator slot == stage slot)
                tc_fence_after();
                const uint32_t sb = base + s * P2_STAGE;
                const uint32_t d_tmem = tbase + s * 256;
                if (st < a.t_steps) {
                    const int N = a.hps * 64;
                    const uint32_t idesc = umma_idesc_bf16(128, N);
                    const uint64_t ad = umma_desc_sw128(sb + P2_SMALL), bd = umma_desc_sw128(sb + P2_BIG);
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        // k-step ks: d-half ks >> 2 (a plane of [rows][128 B]), 32 bytes (ks & 3) inside the 128-byte row
                        const uint64_t ao = (uint64_t)(((ks >> 2) * (128 * 128) + (ks & 3) * 32) >> 4);
                        const uint64_t bo = (uint64_t)(((ks >> 2) * (N * 128) + (ks & 3) * 32) >> 4);
                        umma_bf16_ss_elect(d_tmem, ad + ao, bd + bo, idesc, ks > 0);
                    }
                } else {
                    // student: selector head h of this step = planes ppl h .. ppl h + ppl - 1 (ppl = d_idx / 64), columns 64 h'
                    const int ppl = a.d_idx >> 6, heads = 4 / ppl;
                    const uint32_t idesc = umma_idesc_bf16(128, 64);
                    for (int hh = 0; hh < heads; ++hh)
                        for (int ks = 0; ks < 4 * ppl; ++ks) {
                            const int plane = hh * ppl + (ks >> 2);
                            const uint64_t ad = umma_desc_sw128(sb + P2_BIG + plane * (128 * 128) + (ks & 3) * 32);
                            const uint64_t bd = umma_desc_sw128(sb + P2_SMALL + plane * (64 * 128) + (ks & 3) * 32);
                            umma_bf16_ss_elect(d_tmem + hh * 64, ad, bd, idesc, ks > 0);
                        }
                }
                umma_commit_elect(bar_t_full + 8 * s);
                umma_commit_elect(bar_empty + 8 * s);
            }
    } else if (warp >= 4) {
        // ================================ epilogue (warps 4 .. 11) ================================
        const int lq = warp & 3, qh = (warp - 4) >> 2;
        const int key_l = lq * 32 + lane;                              // this thread's key inside the tile = TMEM lane
        const uint32_t t_lane = tbase + ((uint32_t)(lq * 32) << 16) + qh * 32;
        const int et = threadIdx.x - 128;                              // 0 .. 255 among the epilogue threads
        const float inv_h = 1.f / (float)a.H_q;
        const int bpt = P2_KT / a.blk;                                 // blocks per key tile (8, 4 or 2)
        float acc_d = 0.f, acc_a = 0.f, acc_b = 0.f, acc_c = 0.f;      // lane j: the sums of query qh * 32 + j over this warp's keys
        int n = 0;
        for (int kt = kt_lo; kt < kt_hi; ++kt) {
            // the tile's mask bits of every query of the block: bit u = block kt * bpt + u is in S_q
            if (et < P2_QB) {
                const int b0 = kt * bpt;
                const uint32_t wd = a.mask[(int64_t)(q0 + et) * a.mask_stride + (b0 >> 5)];
                s_bits[(kt & 1) * P2_QB + et] = (wd >> (b0 & 31)) & ((1u << bpt) - 1u);
            }
            float pacc[32], ss[32];
#pragma unroll
            for (int j = 0; j < 32; ++j) { pacc[j] = 0.f; ss[j] = 0.f; }
            for (int st = 0; st < n_steps; ++st, ++n) {
                const int s = n & 1;
                mbar_wait(bar_t_full + 8 * s, (n >> 1) & 1);
                tc_fence_after();
                const uint32_t ta = t_lane + s * 256;
                if (st < a.t_steps) {
                    for (int hh = 0; hh < a.hps; ++hh) {
                        float x[32];
                        tmem_ld32(ta + hh * 64, x);
                        const float4* l4 = reinterpret_cast<const float4*>(s_lse2 + (st * a.hps + hh) * P2_QB + qh * 32);
                        tmem_ld_wait32(x);
#pragma unroll
                        for (int j4 = 0; j4 < 8; ++j4) {
                            const float4 l = l4[j4];                   // (every lane reads the same words: a broadcast)
                            pacc[4 * j4 + 0] += fast_exp2(fmaf(x[4 * j4 + 0], a.scale_log2, -l.x));
                            pacc[4 * j4 + 1] += fast_exp2(fmaf(x[4 * j4 + 1], a.scale_log2, -l.y));
                            pacc[4 * j4 + 2] += fast_exp2(fmaf(x[4 * j4 + 2], a.scale_log2, -l.z));
                            pacc[4 * j4 + 3] += fast_exp2(fmaf(x[4 * j4 + 3], a.scale_log2, -l.w));
                        }
                    }
                } else {
                    const int ppl = a.d_idx >> 6, heads = 4 / ppl, h0 = (st - a.t_steps) * heads;
                    for (int hh = 0; hh < heads; ++hh) {
                        float x[32];
                        tmem_ld32(ta + hh * 64, x);
                        const float4* w4 = reinterpret_cast<const float4*>(s_w + (h0 + hh) * P2_QB + qh * 32);
                        tmem_ld_wait32(x);
#pragma unroll
                        for (int j4 = 0; j4 < 8; ++j4) {
                            const float4 wv = w4[j4];
                            ss[4 * j4 + 0] = fmaf(wv.x, fmaxf(x[4 * j4 + 0], 0.f), ss[4 * j4 + 0]);
                            ss[4 * j4 + 1] = fmaf(wv.y, fmaxf(x[4 * j4 + 1], 0.f), ss[4 * j4 + 1]);
                            ss[4 * j4 + 2] = fmaf(wv.z, fmaxf(x[4 * j4 + 2], 0.f), ss[4 * j4 + 2]);
                            ss[4 * j4 + 3] = fmaf(wv.w, fmaxf(x[4 * j4 + 3], 0.f), ss[4 * j4 + 3]);
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_t_empty + 8 * s);
            }
            // ---- the tile's contributions to the four sums of each query (Eq. 3, Eq. 4; R36: 0 log 0 = 0)
            asm volatile("bar.sync 1, 256;" ::: "memory");              // the tile's mask bits are in shared memory
            const int t = kt * P2_KT + key_l;
            const int blk_in_tile = key_l / a.blk;
            float vd[32], va[32], vb[32], vc[32];
#pragma unroll
            for (int j = 0; j < 32; ++j) {
                const int ql = qh * 32 + j, q = q0 + ql;
                float d = 0.f, A = 0.f, B = 0.f, C = 0.f;
                if (t <= q) {
                    const float pt = pacc[j] * inv_h;
                    const float lps = ss[j] - s_slse[ql];
                    const bool in_s = (s_bits[(kt & 1) * P2_QB + ql] >> blk_in_tile) & 1u;
                    if (in_s) B = __expf(lps);
                    if (pt > 0.f) {
                        const float term = pt * (__logf(pt) - lps);
                        d = term;
                        if (in_s) { A = pt; C = term; }
                    }
                }
                vd[j] = d; va[j] = A; vb[j] = B; vc[j] = C;
            }
            acc_d += warp_transpose_sum(vd, lane);
            acc_a += warp_transpose_sum(va, lane);
            acc_b += warp_transpose_sum(vb, lane);
            acc_c += warp_transpose_sum(vc, lane);
        }
        // ---- the four lane quarters (32 keys each of every tile) of a query half meet in shared memory
        float* mine = s_sum + ((lq * P2_QB) + qh * 32 + lane) * 4;
        mine[0] = acc_d; mine[1] = acc_a; mine[2] = acc_b; mine[3] = acc_c;
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (et < P2_QB) {
            float d = 0.f, A = 0.f, B = 0.f, C = 0.f;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float* v = s_sum + (k * P2_QB + et) * 4;
                d += v[0]; A += v[1]; B += v[2]; C += v[3];
            }
            *reinterpret_cast<float4*>(a.part + ((int64_t)blockIdx.y * a.L + q0 + et) * 4) = make_float4(d, A, B, C);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tbase, 512);
}

// pass 2, last step: the per-chunk sums of every query -> DenseKL (Eq. 3) and SparseKL (Eq. 4)
__global__ void __launch_bounds__(256) pass2_finalize_kernel(const float* __restrict__ part, int kt_chunk, int L,
                                                             float* __restrict__ dense_kl, float* __restrict__ sparse_kl) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= L) return;
    const int n_kt = ((q / P2_QB) * P2_QB + P2_QB + P2_KT - 1) / P2_KT;      // key tiles of the query's block
    const int nch = (n_kt + kt_chunk - 1) / kt_chunk;
    float d = 0.f, A = 0.f, B = 0.f, C = 0.f;
    for (int c = 0; c < nch; ++c) {
        const float4 v = *reinterpret_cast<const float4*>(part + ((int64_t)c * L + q) * 4);
        d += v.x; A += v.y; B += v.z; C += v.w;
    }
    dense_kl[q] = d;
    // Eq. 4: sum_S (p/A) log((p/A) / (s/B)) = C / A - log A + log B
    sparse_kl[q] = A > 0.f ? C / A - __logf(A) + __logf(B) : 0.f;
}

// dst = src * f (the teacher's log-sum-exp from the log2 domain to natural log)
__global__ void scale_copy_kernel(const float* __restrict__ src, float* __restrict__ dst, float f, int64_t n) {
    pdl_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[i] * f;
}

// row q of the selection sees q + 1 tokens
__global__ void iota_len_kernel(int32_t* seq_len, int L) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < L) seq_len[i] = i + 1;
}
// block lists -> bit masks (one warp per query; the mask rows were zeroed by a memset node)
__global__ void list_to_mask_kernel(const int32_t* indices, const int32_t* budgets, int cap, uint32_t* mask, int mask_stride,
                                    int L) {
    const int q = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (q >= L) return;
    const int n = min(budgets[q], cap);
    for (int i = lane; i < n; i += 32) {
        const int b = indices[(int64_t)q * cap + i];
        if (b >= 0) atomicOr(&mask[(int64_t)q * mask_stride + (b >> 5)], 1u << (b & 31));
    }
}

constexpr int P2_KT_CHUNK = 16;                 // key tiles (of 128 keys) per CTA of train_pass2_tc_kernel
struct TrainLayout {
    size_t t_lse2, s_lse, sp_part, p2_part, scores, seq_len, indices, budgets, mask, total;
    int nb_stride, mask_stride, cap, n_b, sp_nch;
};
TrainLayout train_layout(const spot_train_params* p) {
    TrainLayout y;
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    y.n_b = (p->L + p->blk - 1) / p->blk;
    y.nb_stride = (y.n_b + 3) & ~3;
    y.mask_stride = (y.n_b + 31) / 32;
    y.cap = p->top_k < y.n_b ? p->top_k : y.n_b;
    size_t o = 256;
    y.t_lse2 = o; o += up((size_t)p->L * p->H_q * 4);
    y.s_lse = o; o += up((size_t)p->L * 4);
    y.sp_nch = ((p->L + SP_KT - 1) / SP_KT + SP_CHUNK - 1) / SP_CHUNK;
    // (or, on the tensor-core path of the student's pass 1, [L / 64][L] pairs: score_prefill_rows)
    const size_t rows_part = p->L % 64 == 0 ? (size_t)(p->L / 64) * p->L * 8 : 0;
    const size_t chunk_part = (size_t)p->L * y.sp_nch * 8;
    y.sp_part = o; o += up(rows_part > chunk_part ? rows_part : chunk_part);
    y.p2_part = o; o += up((size_t)((p->L + 128 * P2_KT_CHUNK - 1) / (128 * P2_KT_CHUNK)) * p->L * 16);
    y.scores = o; o += up((size_t)p->L * y.nb_stride * 4);
    y.seq_len = o; o += up((size_t)p->L * 4);
    y.indices = o; o += p->indices ? 0 : up((size_t)p->L * y.cap * 4);
    y.budgets = o; o += p->budgets ? 0 : up((size_t)p->L * 4);
    y.mask = o; o += up((size_t)p->L * y.mask_stride * 4);
    y.total = o;
    return y;
}

spot_status check_train(const spot_train_params* p) {
    if (!p || !p->q || !p->k || !p->sel_q || !p->w || !p->sel_k || !p->dense_kl || !p->sparse_kl) return SPOT_ERR_INVALID_ARG;
    if (!aligned16(p->q) || !aligned16(p->k) || !aligned16(p->sel_q) || !aligned16(p->sel_k)) return SPOT_ERR_INVALID_ARG;
    if (p->L <= 0 || p->H_q <= 0 || p->H_kv <= 0 || p->H_q % p->H_kv != 0 || p->H_idx <= 0 || p->d_idx <= 0) return SPOT_ERR_INVALID_ARG;
    if (p->top_k <= 0 || p->sink_blocks < 0 || p->recency_blocks < 0 || p->top_k < p->sink_blocks + p->recency_blocks)
        return SPOT_ERR_INVALID_ARG;
    if (p->k_stride_token < p->D || p->k_stride_token % 8 || p->k_stride_head % 8) return SPOT_ERR_INVALID_ARG;
    if ((p->indices == nullptr) != (p->budgets == nullptr)) return SPOT_ERR_INVALID_ARG;
    const int G = p->H_q / p->H_kv;
    if (p->D != TR_D || p->H_kv > TR_TW || (G != 2 && G != 4 && G != 8 && G != 16)) return SPOT_ERR_UNSUPPORTED;
    if (p->H_idx > 4 || p->d_idx % 16 != 0 || p->d_idx > 128) return SPOT_ERR_UNSUPPORTED;
    if (p->blk != 16 && p->blk != 32 && p->blk != 64) return SPOT_ERR_UNSUPPORTED;
    if ((p->L + p->blk - 1) / p->blk > SEL_MAX_NB) return SPOT_ERR_UNSUPPORTED;
    if (p->indices && p->cap < ((p->L + p->blk - 1) / p->blk < p->top_k ? (p->L + p->blk - 1) / p->blk : p->top_k))
        return SPOT_ERR_INVALID_ARG;
    return SPOT_OK;
}


// pass 2 on the tensor cores: L whole 64-query blocks, H_q <= 32, selector 4 x 64 or 4 x 128
bool pass2_tc_supported(const spot_train_params* p) {
    const int G = p->H_q / p->H_kv;
    return p->L % 64 == 0 && p->H_q <= 32 && p->H_idx == 4 && (p->d_idx == 64 || p->d_idx == 128) &&
           (G == 2 || G == 4 || G == 8 || G == 16) && (p->blk == 16 || p->blk == 32 || p->blk == 64);
}

spot_status launch_pass2_tc(const spot_train_params* p, const TrainArgs& t, cudaStream_t s) {
    Pass2Args a;
    memset(&a, 0, sizeof(a));
    a.t_lse2 = t.t_lse2; a.s_lse = t.s_lse; a.w = p->w; a.mask = t.mask; a.mask_stride = t.mask_stride;
    a.L = p->L; a.H_q = p->H_q; a.G = p->H_q / p->H_kv; a.d_idx = p->d_idx; a.blk = p->blk;
    a.hps = a.G < 4 ? a.G : 4;
    a.t_steps = p->H_q / a.hps; a.s_steps = p->d_idx / 64;
    a.scale_log2 = t.scale_log2;
    a.dense_kl = p->dense_kl; a.sparse_kl = p->sparse_kl;
    a.part = t.p2_part; a.kt_chunk = P2_KT_CHUNK;
    CUtensorMap tm_q, tm_k, tm_sq, tm_sk;
    {   // Q [L][H_q][128] as (64 d, query, head, d-half, 1): a box of 64 queries x hps heads x 2 halves lands as
        // [half][head][query][128 B] = [half][hps * 64 columns][128 B]
        const uint64_t dims[5] = {64, (uint64_t)p->L, (uint64_t)p->H_q, 2, 1};
        const uint64_t strides[4] = {(uint64_t)p->H_q * 256, 256, 128, (uint64_t)p->L * p->H_q * 256};
        const uint32_t box[5] = {64, 64, (uint32_t)a.hps, 2, 1};
        if (!encode_tmap_bf16_sw128(&tm_q, p->q, 5, dims, strides, box)) return SPOT_ERR_CUDA;
    }
    {   // K as (64 d, token, d-half, KV head, 1): a box of 128 keys x 2 halves lands as [half][128 keys][128 B]
        const uint64_t dims[5] = {64, (uint64_t)p->L, 2, (uint64_t)p->H_kv, 1};
        const uint64_t strides[4] = {(uint64_t)p->k_stride_token * 2, 128, (uint64_t)p->k_stride_head * 2,
                                     (uint64_t)p->L * p->H_kv * 256};
        const uint32_t box[5] = {64, 128, 2, 1, 1};
        if (!encode_tmap_bf16_sw128(&tm_k, p->k, 5, dims, strides, box)) return SPOT_ERR_CUDA;
    }
    const uint64_t planes = (uint64_t)4 * p->d_idx / 64, row_bytes = planes * 128;
    {   // selector rows [L][4 x d_idx] as (64 elements = one 128-byte plane, token, plane, 1): four planes per box
        const uint64_t dims[4] = {64, (uint64_t)p->L, planes, 1};
        const uint64_t strides[3] = {row_bytes, 128, (uint64_t)p->L * row_bytes};
        const uint32_t boxq[4] = {64, 64, 4, 1}, boxk[4] = {64, 128, 4, 1};
        if (!encode_tmap_bf16_sw128(&tm_sq, p->sel_q, 4, dims, strides, boxq)) return SPOT_ERR_CUDA;
        if (!encode_tmap_bf16_sw128(&tm_sk, p->sel_k, 4, dims, strides, boxk)) return SPOT_ERR_CUDA;
    }
    static unsigned long long done = 0;
    SPOT_CUDA_TRY(set_max_smem_once(train_pass2_tc_kernel, (int)P2_SMEM, done));
    const int nch = ((p->L + P2_KT - 1) / P2_KT + P2_KT_CHUNK - 1) / P2_KT_CHUNK;
    train_pass2_tc_kernel<<<dim3((unsigned)(p->L / P2_QB), (unsigned)nch), P2_THREADS, P2_SMEM, s>>>(tm_q, tm_k, tm_sq, tm_sk, a);
    SPOT_LAUNCH_CHECK();
    pass2_finalize_kernel<<<(p->L + 255) / 256, 256, 0, s>>>(a.part, a.kt_chunk, p->L, p->dense_kl, p->sparse_kl);
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}

}  // namespace

}  // namespace spot

using namespace spot;

extern "C" size_t spot_train_kl_workspace_bytes(const spot_train_params* p) {
    if (check_train(p) != SPOT_OK) return 0;
    return train_layout(p).total;
}

extern "C" spot_status spot_train_kl(const spot_train_params* p, void* stream) {
    spot_status st = check_train(p);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    const TrainLayout y = train_layout(p);
    if (!p->workspace || p->workspace_bytes < y.total) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)stream;
    if (!aligned16(p->workspace)) return SPOT_ERR_INVALID_ARG;
    char* ws = reinterpret_cast<char*>(p->workspace);
    TrainArgs a;
    memset(&a, 0, sizeof(a));
    a.q = p->q; a.k = p->k; a.k_st = p->k_stride_token; a.k_sh = p->k_stride_head;
    a.sel_q = p->sel_q; a.w = p->w; a.sel_k = p->sel_k;
    a.L = p->L; a.H_q = p->H_q; a.H_kv = p->H_kv; a.G = p->H_q / p->H_kv; a.H_idx = p->H_idx; a.d_idx = p->d_idx; a.blk = p->blk;
    a.scale_log2 = p->sm_scale * 1.4426950408889634f;
    a.t_lse2 = reinterpret_cast<float*>(ws + y.t_lse2);
    a.s_lse = reinterpret_cast<float*>(ws + y.s_lse);
    a.sp_part = reinterpret_cast<float*>(ws + y.sp_part); a.sp_nch = y.sp_nch;
    a.p2_part = reinterpret_cast<float*>(ws + y.p2_part);
    a.blk_scores = reinterpret_cast<float*>(ws + y.scores);
    a.nb_stride = y.nb_stride;
    uint32_t* mask = reinterpret_cast<uint32_t*>(ws + y.mask);
    a.mask = mask; a.mask_stride = y.mask_stride;
    a.dense_kl = p->dense_kl; a.sparse_kl = p->sparse_kl; a.teacher_lse = p->teacher_lse;
    int32_t* seq_len = reinterpret_cast<int32_t*>(ws + y.seq_len);
    int32_t* indices = p->indices ? p->indices : reinterpret_cast<int32_t*>(ws + y.indices);
    int32_t* budgets = p->budgets ? p->budgets : reinterpret_cast<int32_t*>(ws + y.budgets);
    const int cap = p->indices ? p->cap : y.cap;

    const int QPC = 32 / a.G;
    const int grid = (p->L + QPC - 1) / QPC;
    const int smem = TR_TW * TR_STAGES * TR_KSTAGE + TR_STAGES * TR_KT * (p->H_idx * p->d_idx * 2) + 4 * TR_QMAX * TR_KT * 4 +
                     16 * (p->H_idx * p->d_idx * 2);
    static unsigned long long done1 = 0, done2 = 0;
    // (the attribute is set once per device: to the largest geometry, H_idx x d_idx = 4 x 128)
    constexpr int smem_max = TR_TW * TR_STAGES * TR_KSTAGE + TR_STAGES * TR_KT * 1024 + 4 * TR_QMAX * TR_KT * 4 + 16 * 1024;
    SPOT_CUDA_TRY(set_max_smem_once(train_pass_kernel<1>, smem_max, done1));
    SPOT_CUDA_TRY(set_max_smem_once(train_pass_kernel<2>, smem_max, done2));
    // Pass 1.  The teacher's part (the log-sum-exp of every (query, head) row) is flash attention's softmax statistics: when
    // the sequence is whole 64-query blocks it runs on the tcgen05 kernel of the prefill path in its statistics-only form
    // (attn_prefill_tc.cu), and the student's part in a kernel of its own; otherwise both in train_pass_kernel<1>.
    if (p->L % 64 == 0) {
        if ((st = attn_prefill_stats(p->q, p->k, p->k_stride_token, p->k_stride_head, p->L, p->H_q, p->H_kv, p->sm_scale,
                                     a.t_lse2, s)) != SPOT_OK)
            return st;
        if (p->teacher_lse) {
            scale_copy_kernel<<<(unsigned)(((int64_t)p->L * p->H_q + 255) / 256), 256, 0, s>>>(
                a.t_lse2, p->teacher_lse, 0.6931471805599453f, (int64_t)p->L * p->H_q);
            SPOT_LAUNCH_CHECK();
        }
        // the student's part: the tile-score GEMM of the prefill path in its rows form (tcgen05) where its geometry fits,
        // else student_pass1_kernel (mma.sync)
        const bool rows_tc = p->H_idx == 4 && (p->d_idx == 64 || p->d_idx == 128) && (p->blk == 16 || p->blk == 32 || p->blk == 64);
        if (rows_tc) {
            if ((st = score_prefill_rows(p->sel_q, p->w, p->sel_k, p->L, p->H_idx, p->d_idx, p->blk, a.blk_scores, a.nb_stride,
                                         reinterpret_cast<float2*>(a.sp_part), s)) != SPOT_OK)
                return st;
            student_combine_rows_kernel<<<(8 * p->L + 255) / 256, 256, 0, s>>>(reinterpret_cast<const float2*>(a.sp_part), a.s_lse, p->L);
            SPOT_LAUNCH_CHECK();
        } else {
        const int srow = p->H_idx * p->d_idx * 2, stages = 2;
        const int sp_smem = (stages * SP_KT + SP_QPC) * srow;
        static unsigned long long done3 = 0;
        SPOT_CUDA_TRY(set_max_smem_once(student_pass1_kernel, (2 * SP_KT + SP_QPC) * 1024, done3));
        student_pass1_kernel<<<dim3((unsigned)a.sp_nch, (unsigned)((p->L + SP_QPC - 1) / SP_QPC)), SP_THREADS, sp_smem, s>>>(a, stages);
        SPOT_LAUNCH_CHECK();
        student_combine_kernel<<<(p->L + 255) / 256, 256, 0, s>>>(a.sp_part, a.sp_nch, a.s_lse, p->L);
        SPOT_LAUNCH_CHECK();
        }
    } else {
        train_pass_kernel<1><<<grid, TR_THREADS, smem, s>>>(a);
        SPOT_LAUNCH_CHECK();
    }
    iota_len_kernel<<<(p->L + 255) / 256, 256, 0, s>>>(seq_len, p->L);
    SPOT_LAUNCH_CHECK();
    // Eq. 6 per query: the selection kernel in its decode form, one row per query
    spot_select_params sp;
    memset(&sp, 0, sizeof(sp));
    sp.seq_len = seq_len; sp.max_seq_len = p->L; sp.B = p->L; sp.Tq = 1; sp.H_idx = p->H_idx; sp.d_idx = p->d_idx;
    sp.blk = p->blk; sp.q_block = 1; sp.mode = SPOT_MODE_TOPK; sp.top_k = p->top_k; sp.p = 1.0; sp.temperature = 1.0;
    sp.sink_blocks = p->sink_blocks; sp.recency_blocks = p->recency_blocks; sp.kmin_blocks = 0;
    sp.indices = indices; sp.cap = cap; sp.budgets = budgets; sp.nb_stride = y.nb_stride;
    if ((st = run_select(&sp, a.blk_scores, y.nb_stride, 1, y.n_b, nullptr, s)) != SPOT_OK) return st;
    SPOT_CUDA_TRY(cudaMemsetAsync(mask, 0, (size_t)p->L * y.mask_stride * 4, s));
    list_to_mask_kernel<<<(p->L + 7) / 8, 256, 0, s>>>(indices, budgets, cap, mask, y.mask_stride, p->L);
    SPOT_LAUNCH_CHECK();
    if (pass2_tc_supported(p)) return launch_pass2_tc(p, a, s);
    train_pass_kernel<2><<<grid, TR_THREADS, smem, s>>>(a);
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}
