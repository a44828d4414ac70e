// Step a3' on the 5th-generation tensor cores -- block-sparse causal GQA flash attention for chunked prefill
// (Fig. 2): every 64-token query block attends to its own list of selected 64-token key
// blocks; only the diagonal block needs a token-level mask.
//
// Tensor-bound.  Work item = (sequence, query block, KV head, PAIR of 128-row tiles); rows stack the group's query
// heads: row = head_in_group * 64 + query, so one K/V tile in shared memory feeds every head of the group.
// One iteration covers a PAIR of selected key blocks (128 keys; any two blocks of the list, the last pair may be single).
//   warp 0 lane 0 : TMA producer.  Q (two [2 d-halves][128 rows][64] tiles) once, then a 2-stage ring of K pairs and V
//                   pairs ([2 d-halves][128 keys][64], 32 KiB each, 128-byte swizzle; a block is four 8 KiB boxes)
//                   through rank-5 tensor maps built from the caller's element strides.
//   warp 1 lane 0 : tcgen05.mma issuer.  S_t = Q_t K^T (M=128, N=128, 8 k-steps, both operands K-major in shared
//                   memory) into TMEM; O_t += P_t V (M=128, N=128, 8 k-steps) with P_t read from TENSOR MEMORY (packed
//                   BF16 over the start of S_t) and V used as an MN-major B operand exactly as TMA wrote it (no
//                   transpose).  Descriptors are built once and advanced by constants: the lone issuing thread has
//                   nobody to hide its instruction latencies.  The two tiles ping-pong:
//                       PV0(n)  QK0(n+1)  |  PV1(n)  QK1(n+1)  | ...
//   warps 4-7, 8-11: softmax of tile 0 / tile 1, one thread per row (TMEM lane = row).  One optimistic pass over the 128
//                   logits (exp against the stale max while the new max is found; redone only when a rescale is
//                   due), log2-domain online softmax (scale and max-subtraction fused
//                   into one FFMA per element) with a LAZY rescale of the TMEM-resident O (only when a row's max grows
//                   by more than 2^8 since the last rescale: P stays <= 256, l and O use the same stale max, so the
//                   result is exact), P rounded to BF16 and stored back to TMEM (tcgen05.st), mbarrier hand-off.
//                   Epilogue: O / l -> BF16, 256 B per row, optional LSE.  (Named barriers that forced the two tiles'
//                   exp sections to alternate were measured and dropped: 1069 vs 1096 TFLOP/s without.)
// TMEM: S_0 | S_1 | O_0 | O_1 = 128 + 128 + 128 + 128 columns (all 512).  Grid: (tile pair, query block heaviest-first,
// KV head) with the KV head slowest, so the CTAs in flight share one head's K/V in L2 (DRAM reads 25 GB -> 0.8 GB).
// History (cfg5, TFLOP/s): mma.sync 328 -> tcgen05 SS 789 -> fused FFMA 805 -> P in TMEM 826 -> hoisted descriptors
// 887 -> head-slowest grid 982 -> 128 keys per iteration 1016 -> optimistic single-pass softmax 1069 -> no ordering barriers 1096
// -> converged issuer warp with an elected lane 1105.  (Round 2, measured and dropped: 2 / 3 / 4 of every 8 exponentials through a
// Cody-Waite + cubic polynomial on the FMA / ALU pipes instead of MUFU.EX2: 1065 / 1039 / 993 -- the softmax warps are
// bound by issue slots, not by the 16 MUFU lanes.  Also measured and dropped: P handed to the issuer in HALVES of 64 keys, each
// a softmax step of its own with its own barrier, so that PV of the first half runs under the exponentials of the second:
// 954 against 1100 TFLOP/s at cfg5 -- twice the hand-offs per tile cost more than the overlap returns (and its parity was not green yet: a few rows off); one issuer warp PER TILE (each tile's chain on a warp of its own instead of one
// warp alternating between the tiles; parity green): 916 TFLOP/s -- the fixed PV0 QK0 | PV1 QK1 order of the single issuer is
// what keeps the two tiles half an iteration apart.)
#include "common.cuh"
#include "tc100.cuh"

#include <string.h>

namespace spot {

namespace {

constexpr int TA_STAGES = 2;
constexpr int TA_THREADS = 12 * 32;
constexpr uint32_t TA_Q_TILE = 2 * 128 * 128;          // 32 KiB: [2 halves][128 rows][128 B]
constexpr uint32_t TA_KV_TILE = 2 * 128 * 128;         // 32 KiB: [2 halves][128 keys = a PAIR of key blocks][128 B]
constexpr uint32_t TA_BLK_BYTES = 2 * 64 * 128;        // 16 KiB of K (or V) per 64-key block
constexpr uint32_t TA_SMEM_TILES = 2 * TA_Q_TILE + TA_STAGES * 2 * TA_KV_TILE;   // 192 KiB
constexpr uint32_t TA_SMEM_BYTES = 1024 + TA_SMEM_TILES + 256;
constexpr float TA_RESCALE_THRESHOLD = 8.0f;           // log2 units

struct TcAttnArgs {
    const int32_t* indices;      // [B * n_qb][cap]; nullptr: every causally visible block
    const int32_t* page_table;   // nullptr: contiguous K/V; else page pools (f3, R32): [B][pt_stride] physical pages
    int pt_stride, page_tokens;  // page_tokens % 64 == 0: a 64-token block never straddles pages
    const int32_t* budgets;
    int cap;
    int Tq, n_qb, H_q, H_kv, G;
    int n_pairs, n_rows;         // grid.x = n_rows * n_pairs: pairs of 128-row tiles per (row, KV head); rows = B * n_qb
    int qb_start;                // q_start / 64
    int blk;                     // key block size of the index lists: 64, or 16 (f3: a 128-key tile gathers 8 list entries)
    float scale_log2;
    uint16_t* out;               // [B][Tq][H_q][128]
    float* lse;                  // optional [B][Tq][H_q]
    float* lse2;                 // STATS form: [B][Tq][H_q] log2-domain log-sum-exp of the scaled logits
#ifdef SPOT_TRACE
    long long* trace;            // development builds only: [12 roles][512 iterations] clock64 of one CTA
#endif
};
#ifdef SPOT_TRACE
long long* g_ta_trace = nullptr;
#define TA_STAMP(role, it) do { if (a.trace && blockIdx.x == 0 && blockIdx.z == 0 && (it) < 512) a.trace[(role) * 512 + (it)] = clock64(); } while (0)
#else
#define TA_STAMP(role, it) do { } while (0)
#endif

template <int BLK, bool STATS = false>
                         // BLK: key block size of the index lists: 64, or 16 (f3) -- a compile-time constant: the softmax warps
                         // are a co-bound of this kernel and the 64-token form must not pay for the per-16-key causal limits.
                         // STATS (f4, train_kl.cu): only the softmax statistics -- the log-sum-exp of every (query, head) row,
                         // log2 domain, to a.lse2 -- no V, no P, no PV product, no output: the teacher pass 1 of Eq. 1
__global__ void __launch_bounds__(TA_THREADS, 1) attn_prefill_tc_kernel(const __grid_constant__ CUtensorMap tm_q,
                                                                        const __grid_constant__ CUtensorMap tm_k,
                                                                        const __grid_constant__ CUtensorMap tm_v,
                                                                        const TcAttnArgs a) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* smem = smem_raw + (base - smem_u32(smem_raw));
    const uint32_t q_smem = base;                                        // 2 x 32 KiB
    const uint32_t kv_smem = base + 2 * TA_Q_TILE;                       // stages x (K 16 KiB, V 16 KiB)
    const uint32_t misc = base + TA_SMEM_TILES;
    const uint32_t bar_q_full = misc;
    const uint32_t bar_k_full = misc + 8;                // [TA_STAGES]
    const uint32_t bar_v_full = misc + 40;               // [TA_STAGES]
    const uint32_t bar_kv_empty = misc + 72;             // [TA_STAGES]
    const uint32_t bar_s_full = misc + 104;              // [2]
    const uint32_t bar_p_full = misc + 120;              // [2]
    const uint32_t bar_o_done = misc + 136;              // [2]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + TA_SMEM_TILES + 160);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // launch order: x (tile pair) fastest, then y (query block, heaviest = latest first), KV head slowest -- the CTAs in
    // flight at any time share ONE head's K/V (32 MiB at L = 64K, L2-resident) instead of all eight heads' (256 MiB)
    // (tile pair and row share blockIdx.x -- up to 2^31 - 1 -- so that B * Tq / 64 is not bound by the 65535 of y / z)
    const int pair = (int)(blockIdx.x % (unsigned)a.n_pairs), hk = blockIdx.z;
    const int rowz = a.n_rows - 1 - (int)(blockIdx.x / (unsigned)a.n_pairs);
    const int b = rowz / a.n_qb, i = rowz - b * a.n_qb;
    const int G = a.G;
    const int qb_abs = a.qb_start + i;
    const bool two = (2 * pair + 1) * 2 < G;                             // does the pair's second tile have live rows?

    if (threadIdx.x == 0) {
        mbar_init(bar_q_full, 1);
        for (int s = 0; s < TA_STAGES; ++s) {
            mbar_init(bar_k_full + 8 * s, 1);
            mbar_init(bar_v_full + 8 * s, 1);
            mbar_init(bar_kv_empty + 8 * s, 1);
        }
        for (int t = 0; t < 2; ++t) {
            mbar_init(bar_s_full + 8 * t, 1);
            mbar_init(bar_p_full + 8 * t, 128);
            mbar_init(bar_o_done + 8 * t, 1);
        }
        mbar_fence_init();
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
    }
    if (warp == 2) tmem_alloc(misc + 160, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tbase = *tmem_slot;
    pdl_wait();
    pdl_launch_dependents();

    const int budget = a.indices ? max(0, min(a.budgets[rowz], a.cap)) : (qb_abs + 1) * (64 / BLK);
    const int32_t* idx = a.indices ? a.indices + (int64_t)rowz * a.cap : nullptr;
    // one tile of the loop = up to GROUP visible list entries = up to 128 keys (2 x 64 or 8 x 16)
    constexpr int blk = BLK, GROUP = 128 / BLK;
    constexpr int blk_shift = BLK == 16 ? 2 : 0;         // list entry -> 64-token block: j >> blk_shift
    auto block_of = [&](int it) -> int { return idx ? idx[it] : it; };
    auto visible = [&](int j) -> bool { return j >= 0 && (j >> blk_shift) <= qb_abs; };
    // where key block j lives: (token coordinate, outermost coordinate) of the K / V tensor maps -- (64 j, b) for
    // contiguous caches, (offset inside the page, physical page) for page pools
    const int32_t* ptab = a.page_table ? a.page_table + (int64_t)b * a.pt_stride : nullptr;
    auto place = [&](int j, int& tok, int& outer) {
        tok = j * blk;
        outer = b;
        if (ptab) {
            const int lp = tok / a.page_tokens;
            outer = ptab[lp];
            tok -= lp * a.page_tokens;
        }
    };

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            mbar_arrive_expect_tx(bar_q_full, two ? 2 * TA_Q_TILE : TA_Q_TILE);
            for (int t = 0; t < (two ? 2 : 1); ++t)
                tma_load_5d(q_smem + t * TA_Q_TILE, &tm_q, bar_q_full, 0, i * 64, hk * G + (2 * pair + t) * 2, 0, b);
            // one ring stage = a PAIR of visible key blocks (any two, they need not be adjacent): K pair, then V pair,
            // each [2 d-halves][128 keys][128 B]; a block is four 8 KiB boxes (K/V x d-half)
            int n = 0, it = 0;
            const uint32_t ent_bytes = (uint32_t)blk * 128u;                  // one d-half of one list entry
            while (true) {
                // (the page-table lookups are issued before the wait for the ring slot, which hides them)
                int tok[8], outer[8], ne = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    tok[u] = outer[u] = 0;
                    if (u < GROUP)
                        while (it < budget) {
                            const int j = block_of(it++);
                            if (visible(j)) { place(j, tok[u], outer[u]); ++ne; break; }
                        }
                }
                if (ne == 0) break;
                const int s = n % TA_STAGES;
                mbar_wait(bar_kv_empty + 8 * s, ((n / TA_STAGES) & 1) ^ 1);
                const uint32_t ks = kv_smem + s * 2 * TA_KV_TILE;
                const uint32_t bytes = (uint32_t)ne * 2u * ent_bytes;
                mbar_arrive_expect_tx(bar_k_full + 8 * s, bytes);
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (u < ne)
                        for (int hf = 0; hf < 2; ++hf)
                            tma_load_5d(ks + hf * (128 * 128) + u * ent_bytes, &tm_k, bar_k_full + 8 * s, 0, tok[u], hf, hk,
                                        outer[u]);
                if constexpr (!STATS) {
                    mbar_arrive_expect_tx(bar_v_full + 8 * s, bytes);
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (u < ne)
                            for (int hf = 0; hf < 2; ++hf)
                                tma_load_5d(ks + TA_KV_TILE + hf * (128 * 128) + u * ent_bytes, &tm_v, bar_v_full + 8 * s, 0,
                                            tok[u], hf, hk, outer[u]);
                }
                ++n;
            }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer ================================
        // The whole warp runs this converged; one ELECTED lane issues (tc100.cuh, umma_*_elect): under `if (lane == 0)`
        // every tcgen05.mma sat in an ELECT / BRA.U.ANY loop of its own and cost the lone thread 70-130 cycles.
        {
            constexpr uint32_t idesc_pv = umma_idesc_bf16(128, 128) | UMMA_B_MN_MAJOR;
            int nv = 0;
            for (int it = 0; it < budget; ++it) nv += visible(block_of(it)) ? 1 : 0;
            const int np = (nv + GROUP - 1) / GROUP;     // iterations: tiles of up to 128 keys (the last may be short)
            auto keys_of = [&](int n) -> int { return min(GROUP, nv - n * GROUP) * blk; };   // keys of tile n: a multiple of 16
            // Descriptors are built
            // once and advanced by compile-time constants (the start-address field is the low 14 bits, in 16-byte
            // units), so each tcgen05.mma costs two integer adds, not a dozen dependent ones.
            const uint64_t qd[2] = {umma_desc_sw128(q_smem), umma_desc_sw128(q_smem + TA_Q_TILE)};
            auto qk = [&](int t, uint64_t kd, int nkeys) {     // S_t = Q_t K^T over nkeys keys (N = nkeys)
                const uint32_t idesc = umma_idesc_bf16(128, nkeys);
#pragma unroll
                for (int kk = 0; kk < 8; ++kk)
                    umma_bf16_ss_elect(tbase + t * 128, qd[t] + (uint64_t)(((kk >> 2) * (128 * 128) + (kk & 3) * 32) >> 4),
                                 kd + (uint64_t)(((kk >> 2) * (128 * 128) + (kk & 3) * 32) >> 4), idesc, kk > 0);
                umma_commit_elect(bar_s_full + 8 * t);
            };
            auto pv = [&](int t, uint64_t vd, bool acc, int nkeys) {   // O_t += P_t V over nkeys keys: one k-step per 16 keys
#pragma unroll
                for (int kk = 0; kk < 8; ++kk)
                    if (kk * 16 < nkeys)
                        umma_bf16_ts_elect(tbase + 256 + t * 128, tbase + t * 128 + kk * 8, vd + (uint64_t)((kk * 2048) >> 4),
                                     idesc_pv, acc || kk > 0);
                umma_commit_elect(bar_o_done + 8 * t);
            };
            if (np > 0) {
                mbar_wait(bar_q_full, 0);
                mbar_wait(bar_k_full, 0);
                tc_fence_after();
                {
                    const uint64_t kd0 = umma_desc_sw128(kv_smem);
                    qk(0, kd0, keys_of(0));
                    if (two) qk(1, kd0, keys_of(0));
                }
                for (int n = 0; n < np; ++n) {
                    const int s = n % TA_STAGES, s1 = (n + 1) % TA_STAGES;
                    const uint64_t vd = umma_desc_sw128_mn(kv_smem + s * 2 * TA_KV_TILE + TA_KV_TILE, 128 * 128, 1024);
                    const uint64_t kd1 = umma_desc_sw128(kv_smem + s1 * 2 * TA_KV_TILE);
                    const bool more = n + 1 < np;
                    const int nk0 = keys_of(n), nk1 = more ? keys_of(n + 1) : 0;
                    if constexpr (!STATS) mbar_wait(bar_v_full + 8 * s, (n / TA_STAGES) & 1);
                    if (more) mbar_wait(bar_k_full + 8 * s1, ((n + 1) / TA_STAGES) & 1);
                    mbar_wait(bar_p_full, n & 1);                       // P_0(n) written, S_0 consumed, O_0 rescaled
                    if (lane == 0) TA_STAMP(0, n);
                    tc_fence_after();
                    if constexpr (!STATS) pv(0, vd, n > 0, nk0);
                    if (more) qk(0, kd1, nk1);
                    if (lane == 0) TA_STAMP(1, n);
                    if (two) {
                        mbar_wait(bar_p_full + 8, n & 1);
                        if (lane == 0) TA_STAMP(2, n);
                        tc_fence_after();
                        if constexpr (!STATS) pv(1, vd, n > 0, nk0);
                        if (more) qk(1, kd1, nk1);
                        if (lane == 0) TA_STAMP(3, n);
                    }
                    umma_commit_elect(bar_kv_empty + 8 * s);                  // K(n), V(n) no longer read
                }
            }
        }
    } else if (warp >= 4) {
        // ================================ softmax + epilogue ================================
        const int t = (warp - 4) >> 2;                    // tile of the pair
        const int lq = warp & 3;                          // TMEM lane quarter this warp may access
        if (t == 0 || two) {
            const int r = lq * 32 + lane;                 // row of the tile = TMEM lane
            const int hg = (2 * pair + t) * 2 + (r >> 6); // head in group
            const int ql = r & 63;                        // query in block
            const bool live = hg < G;
            const uint32_t t_s = tbase + ((uint32_t)(lq * 32) << 16) + t * 128;
            const uint32_t t_o = tbase + ((uint32_t)(lq * 32) << 16) + 256 + t * 128;
            float m_used = -INFINITY, l = 0.f;
            int n = 0, it = 0;
            while (true) {
                // this iteration's tile: up to GROUP visible list entries (the last tile may be short)
                int jj[8], ne = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) {                   // (static indices: jj[] stays in registers)
                    jj[u] = -1;
                    if (u < GROUP)
                        while (it < budget) {
                            const int j = block_of(it++);
                            if (visible(j)) { jj[u] = j; ++ne; break; }
                        }
                }
                if (ne == 0) break;
                const int nkeys = ne * blk, nh = (nkeys + 63) >> 6;
                // 16-token blocks: causal limit of every 16-key group u of the tile -- key e of the group is visible iff
                // e <= lim(u) (15: the whole group, the usual case; -1: none -- a group past the end of a short tile, or a
                // block that lies wholly in this row's future although the query block as a whole may see it); packed, byte
                // u of lim_pk = lim(u) + 1, so that a loop variable can pick its group without indexing jj[].
                // 64-token blocks: only the diagonal block needs a mask (key e visible iff e <= ql).
                unsigned long long lim_pk = 0ull;
                if constexpr (BLK == 16) {
                    const int q_tok = qb_abs * 64 + ql;
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        int lim = -1;
                        if (u < ne) lim = max(min(15, q_tok - jj[u] * 16), -1);
                        lim_pk |= (unsigned long long)(lim + 1) << (8 * u);
                    }
                }
                auto lim_of = [&](int u) -> int { return (int)((lim_pk >> (8 * u)) & 0xffull) - 1; };
                mbar_wait(bar_s_full + 8 * t, n & 1);
                if (lq == 0 && lane == 0) TA_STAMP(4 + 4 * t, n);
                tc_fence_after();
                // Optimistic single pass: exp2 against the STALE max while the row max of this tile is being found (sm_scale
                // > 0: max on the raw logits; scale and max-subtraction are one FFMA).  P = exp2(scale x - m) rounded to
                // BF16 waits in registers.  Only if some row's max grew by more than 2^8 since its last rescale (always
                // in the first iteration, rarely later) is the tile redone after rescaling O -- P stays <= 256, and l
                // and O always use the same max, so the result is exact.
                uint32_t pk[64];
                float ps0 = 0.f, ps1 = 0.f, mx = -INFINITY;
                {
                    const float neg_m = (m_used == -INFINITY) ? 0.f : -m_used;    // (a row that has seen no key yet)
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        if (hf < nh) {
                            float x[64];
                            {
                                float d0[16], d1[16], d2[16], d3[16];
                                const uint32_t ta = t_s + hf * 64;
                                tmem_ld16(ta, d0); tmem_ld16(ta + 16, d1); tmem_ld16(ta + 32, d2); tmem_ld16(ta + 48, d3);
                                tmem_ld_wait();
#pragma unroll
                                for (int e = 0; e < 16; ++e) { x[e] = d0[e]; x[16 + e] = d1[e]; x[32 + e] = d2[e]; x[48 + e] = d3[e]; }
                            }
                            if constexpr (BLK == 16) {
#pragma unroll
                                for (int g4 = 0; g4 < 4; ++g4) {
                                    const int lim = lim_of(hf * 4 + g4);
                                    if (lim < 15) {
#pragma unroll
                                        for (int e = 0; e < 16; ++e)
                                            if (e > lim) x[g4 * 16 + e] = -INFINITY;
                                    }
                                }
                            } else if (jj[hf] == qb_abs) {
#pragma unroll
                                for (int e = 0; e < 64; ++e)
                                    if (e > ql) x[e] = -INFINITY;
                            }
                            float mxa = fmax3(x[0], x[1], x[2]), mxb = fmax3(x[3], x[4], x[5]);
#pragma unroll
                            for (int e = 6; e < 62; e += 4) { mxa = fmax3(mxa, x[e], x[e + 1]); mxb = fmax3(mxb, x[e + 2], x[e + 3]); }
                            mx = fmaxf(mx, fmax3(fmaxf(mxa, mxb), x[62], x[63]));
#pragma unroll
                            for (int e = 0; e < 64; e += 2) {
                                const float p0 = fast_exp2(fmaf(x[e], a.scale_log2, neg_m));
                                const float p1 = fast_exp2(fmaf(x[e + 1], a.scale_log2, neg_m));
                                ps0 += p0;
                                ps1 += p1;
                                pk[hf * 32 + (e >> 1)] = pack_bf16x2(p0, p1);
                            }
                        }
                    }
                }
                if (lq == 0 && lane == 0) TA_STAMP(5 + 4 * t, n);
                mx *= a.scale_log2;
                const bool need = mx > m_used + TA_RESCALE_THRESHOLD;       // (true for a row's first visible key: m_used = -inf)
                if (__any_sync(0xffffffffu, need)) {                         // warp-uniform: tcgen05.ld/st are collective
                    const float m_new = need ? mx : m_used;
                    const float alpha = (m_used == -INFINITY) ? 0.f : fast_exp2(m_used - m_new);   // 1 when !need
                    l *= alpha;
                    m_used = m_new;
                    if (!STATS && n > 0) {
                        mbar_wait(bar_o_done + 8 * t, (n - 1) & 1);          // PV(n-1) has landed in O_t
                        tc_fence_after();
#pragma unroll
                        for (int cb = 0; cb < 8; ++cb) {
                            float o[16];
                            tmem_ld16(t_o + cb * 16, o);
                            tmem_ld_wait();
#pragma unroll
                            for (int e = 0; e < 16; ++e) o[e] *= alpha;
                            tmem_st16(t_o + cb * 16, o);
                        }
                        tmem_st_wait();
                    }
                    // redo the tile against the new max (S_t is still intact: P has not been stored yet)
                    ps0 = ps1 = 0.f;
                    const float neg_m = (m_used == -INFINITY) ? 0.f : -m_used;
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        if (hf < nh) {
#pragma unroll 1
                            for (int c16 = 0; c16 < 4; ++c16) {
                                float d[16];
                                tmem_ld16(t_s + hf * 64 + c16 * 16, d);
                                tmem_ld_wait();
                                const int lim = BLK == 16 ? lim_of(hf * 4 + c16) : (jj[hf] == qb_abs ? ql - c16 * 16 : 15);
#pragma unroll
                                for (int e = 0; e < 16; e += 2) {
                                    const float x0 = (e > lim) ? -INFINITY : d[e];
                                    const float x1 = (e + 1 > lim) ? -INFINITY : d[e + 1];
                                    const float p0 = fast_exp2(fmaf(x0, a.scale_log2, neg_m));
                                    const float p1 = fast_exp2(fmaf(x1, a.scale_log2, neg_m));
                                    ps0 += p0;
                                    ps1 += p1;
                                    const uint32_t w = pack_bf16x2(p0, p1);
                                    // pk[hf * 32 + c16 * 8 + e / 2] with c16 a loop variable: select statically
#pragma unroll
                                    for (int q = 0; q < 4; ++q)
                                        if (q == c16) pk[hf * 32 + q * 8 + (e >> 1)] = w;
                                }
                            }
                        }
                    }
                }
                // P goes back to tensor memory over the start of S_t: columns 32 hf .. +31 hold the 64 keys of block hf
                // (QK_t(n+1), which rewrites S_t, is issued after PV_t(n) and the tensor pipe runs them in order)
                // (16 columns = 32 keys per store; a short tile stores only what PV will read)
                if (lq == 0 && lane == 0) TA_STAMP(6 + 4 * t, n);
                if constexpr (!STATS) {
                    tmem_st16u(t_s, pk);
                    if (nkeys > 32) tmem_st16u(t_s + 16, pk + 16);
                    if (nkeys > 64) tmem_st16u(t_s + 32, pk + 32);
                    if (nkeys > 96) tmem_st16u(t_s + 48, pk + 48);
                    tmem_st_wait();
                }
                l += ps0 + ps1;
                tc_fence_before();                                   // (STATS: S_t has been read, the next QK^T may overwrite it)
                mbar_arrive(bar_p_full + 8 * t);
                if (lq == 0 && lane == 0) TA_STAMP(7 + 4 * t, n);
                ++n;
            }
            const int q_row = i * 64 + ql;
            const int h = hk * G + hg;
            if constexpr (STATS) {
                // log2-domain log-sum-exp of the row (every query sees at least its own key: l > 0)
                if (live) a.lse2[((int64_t)b * a.Tq + q_row) * a.H_q + h] = l > 0.f ? m_used + log2f(l) : -INFINITY;
            } else {
            // epilogue: O / l -> BF16
            uint16_t* orow = a.out + (((int64_t)b * a.Tq + q_row) * a.H_q + h) * 128;
            if (n > 0) {
                mbar_wait(bar_o_done + 8 * t, (n - 1) & 1);
                tc_fence_after();
            }
            const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
            for (int cb = 0; cb < 8; ++cb) {
                float o[16];
                if (n > 0) {
                    tmem_ld16(t_o + cb * 16, o);
                    tmem_ld_wait();
                } else {
#pragma unroll
                    for (int e = 0; e < 16; ++e) o[e] = 0.f;
                }
                if (live) {
                    uint4 v0, v1;
                    v0.x = pack_bf16x2(o[0] * inv, o[1] * inv);   v0.y = pack_bf16x2(o[2] * inv, o[3] * inv);
                    v0.z = pack_bf16x2(o[4] * inv, o[5] * inv);   v0.w = pack_bf16x2(o[6] * inv, o[7] * inv);
                    v1.x = pack_bf16x2(o[8] * inv, o[9] * inv);   v1.y = pack_bf16x2(o[10] * inv, o[11] * inv);
                    v1.z = pack_bf16x2(o[12] * inv, o[13] * inv); v1.w = pack_bf16x2(o[14] * inv, o[15] * inv);
                    *reinterpret_cast<uint4*>(orow + cb * 16) = v0;
                    *reinterpret_cast<uint4*>(orow + cb * 16 + 8) = v1;
                }
            }
            if (a.lse && live)
                a.lse[((int64_t)b * a.Tq + q_row) * a.H_q + h] =
                    l > 0.f ? (m_used + log2f(l)) * 0.6931471805599453f : -INFINITY;
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tbase, 512);
}

// rank-5 map of a [..][rows][..][128] BF16 tensor as (64 d, rows, 2 d-halves, dim3, dim4): a box of R rows lands in
// shared memory as [2 halves][R][128 B] (K-major 128-byte-swizzled operand tiles).
bool make_map(CUtensorMap* m, const void* base, uint64_t rows, uint64_t row_stride_elems, uint64_t n3,
              uint64_t stride3_elems, uint64_t n4, uint64_t stride4_elems, uint32_t box_rows, uint32_t box3) {
    const uint64_t dims[5] = {64, rows, 2, n3, n4};
    const uint64_t strides[4] = {row_stride_elems * 2, 128, stride3_elems * 2, stride4_elems * 2};
    const uint32_t box[5] = {64, box_rows, 1, box3, 1};          // one d-half per box
    return encode_tmap_bf16_sw128(m, base, 5, dims, strides, box);
}

}  // namespace

// Q [B][Tq][H_q][128]; K/V with element strides; see attn_prefill.cu for the argument checks (already done).
// lse2 != nullptr: the STATS form (blk 64, no page table; p->v, p->out, p->lse are not used).
static spot_status attn_prefill_tc_launch(const spot_attn_params* p, float* lse2, cudaStream_t stream) {
    TcAttnArgs a;
    a.indices = p->indices; a.budgets = p->budgets; a.cap = p->cap;
    a.Tq = p->Tq; a.n_qb = p->Tq / 64; a.H_q = p->H_q; a.H_kv = p->H_kv; a.G = p->H_q / p->H_kv;
    a.qb_start = p->q_start / 64;
    a.blk = p->blk;
    a.scale_log2 = p->sm_scale * 1.4426950408889634f;
    a.out = p->out; a.lse = p->lse; a.lse2 = lse2;
#ifdef SPOT_TRACE
    a.trace = g_ta_trace;
#endif
    const bool stats = lse2 != nullptr;
    if (stats && (p->blk != 64 || p->page_table)) return SPOT_ERR_UNSUPPORTED;
    CUtensorMap tm_q, tm_k, tm_v;
    // Q as (64 d, query, head, d-half, batch): a box of 64 queries x 2 heads x 2 halves lands as
    // [half][head][query][128 B] = [half][128 rows][128 B], row = head * 64 + query.
    {
        const uint64_t dims[5] = {64, (uint64_t)p->Tq, (uint64_t)p->H_q, 2, (uint64_t)p->B};
        const uint64_t strides[4] = {(uint64_t)p->H_q * 128 * 2, 128 * 2, 128, (uint64_t)p->Tq * p->H_q * 128 * 2};
        const uint32_t box[5] = {64, 64, 2, 2, 1};       // -> [half][head][query][128 B] = [half][128 rows][128 B]
        if (!encode_tmap_bf16_sw128(&tm_q, p->q, 5, dims, strides, box)) return SPOT_ERR_CUDA;
    }
    // contiguous caches: (.., token < q_start + Tq, .., head, batch); page pools: (.., token inside a page, .., head,
    // page) -- the pool's size is not part of the ABI, the page coordinate is bounded by what 2^22 pages would hold
    a.page_table = p->page_table; a.pt_stride = p->page_table_stride; a.page_tokens = p->page_tokens;
    const uint64_t n_tok = p->page_table ? (uint64_t)p->page_tokens : (uint64_t)p->q_start + p->Tq;
    const uint64_t n_outer = p->page_table ? ((uint64_t)1 << 22) : (uint64_t)p->B;
    if (!make_map(&tm_k, p->k, n_tok, (uint64_t)p->kv_stride_token, (uint64_t)p->H_kv, (uint64_t)p->kv_stride_head,
                  n_outer, (uint64_t)p->kv_stride_batch, (uint32_t)p->blk, 1))
        return SPOT_ERR_CUDA;
    if (!make_map(&tm_v, stats ? p->k : p->v, n_tok, (uint64_t)p->kv_stride_token, (uint64_t)p->H_kv, (uint64_t)p->kv_stride_head,
                  n_outer, (uint64_t)p->kv_stride_batch, (uint32_t)p->blk, 1))
        return SPOT_ERR_CUDA;
    static unsigned long long smem_attr_done[3] = {0, 0, 0};
    auto kernel = stats ? attn_prefill_tc_kernel<64, true>
                        : (p->blk == 16 ? attn_prefill_tc_kernel<16, false> : attn_prefill_tc_kernel<64, false>);
    SPOT_CUDA_TRY(set_max_smem_once(kernel, (int)TA_SMEM_BYTES, smem_attr_done[stats ? 2 : (p->blk == 16)]));
    const int n_mt = (a.G * 64 + 127) / 128;
    a.n_pairs = (n_mt + 1) / 2;
    a.n_rows = p->B * a.n_qb;
    if ((int64_t)a.n_pairs * a.n_rows > 0x7fffffff || p->H_kv > 65535) return SPOT_ERR_UNSUPPORTED;
    dim3 grid((unsigned)(a.n_pairs * a.n_rows), 1u, (unsigned)p->H_kv);
    SPOT_CUDA_TRY(launch_pdl(kernel, grid, dim3(TA_THREADS), (size_t)TA_SMEM_BYTES, stream, tm_q, tm_k, tm_v, a));
    return SPOT_OK;
}

spot_status attn_prefill_tc(const spot_attn_params* p, cudaStream_t stream) { return attn_prefill_tc_launch(p, nullptr, stream); }

// f4 (train_kl.cu): lse2[q][h] = log2 sum_{t <= q} 2^(scale_log2 q_h . k_{g(h), t}) of ONE sequence of L tokens (L % 64 == 0),
// dense causal -- pass 1 of the teacher distribution (Eq. 1) on the tensor cores.
spot_status attn_prefill_stats(const uint16_t* q, const uint16_t* k, int64_t k_stride_token, int64_t k_stride_head, int L,
                               int H_q, int H_kv, float sm_scale, float* lse2, cudaStream_t stream) {
    if (L <= 0 || L % 64 != 0 || !lse2) return SPOT_ERR_INVALID_ARG;
    spot_attn_params p;
    memset(&p, 0, sizeof(p));
    p.q = q; p.k = k; p.v = k;
    p.kv_stride_batch = (int64_t)L * H_kv * 128; p.kv_stride_token = k_stride_token; p.kv_stride_head = k_stride_head;
    p.B = 1; p.Tq = L; p.q_start = 0; p.H_q = H_q; p.H_kv = H_kv; p.D = 128; p.blk = 64; p.sm_scale = sm_scale;
    return attn_prefill_tc_launch(&p, lse2, stream);
}

}  // namespace spot

#ifdef SPOT_TRACE
extern "C" void spot_debug_set_ta_trace(void* dev_buf) { spot::g_ta_trace = (long long*)dev_buf; }
#endif
