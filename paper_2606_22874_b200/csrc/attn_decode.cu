// Step a3 -- block-sparse GQA flash-decode over the selected 64-token KV blocks (PAPER.md:47 Fig. 2, :71), and the
// dense comparator (every block) from the same code.
//
// HBM-bound: 32 KiB of K+V per (selected block, KV head), 4-8 flop/B.  The work is the flat list of units
// (sequence, KV head, position in that sequence's index list), U = H_kv * sum_b budget_b of them, and it is cut
// stream-K style into gridDim.x equal contiguous ranges, one per persistent CTA (2 CTAs per SM): every CTA streams the
// same number of bytes whatever the budgets are (config 4's 8..512-block mix included) and the whole grid is one wave.
// A CTA's range touches one segment (sequence, KV head) or a few; for each it keeps a private online-softmax state
// and writes ONE unnormalised partial (m, l, O) -- <= gridDim.x + B*H_kv partials in total (slot = CTA + segment
// index, unique because the (CTA, segment) pairs form a staircase), a few hundred KiB instead of one per 8 blocks.
// Inside the CTA every warp runs its OWN cp.async ring over its 16-token quarter of each block (8 KiB of K+V per
// stage, zero CTA-wide barriers in the main loop) and feeds ldmatrix -> mma.sync m16n8k16 with the G = H_q/H_kv query
// heads of the group as the (padded) M = 16 rows.  M is tiny here, so this is mma.sync territory, not tcgen05: the
// tensor pipe needs < 15 % of the time the HBM stream takes.  A second small kernel merges each (sequence, head)'s
// partials (log-sum-exp) and writes BF16.
//
// Two next-row options ride on the same loop: with 16-token blocks (blk == 16) a unit is four
// consecutive entries of the index list, one per warp (a short last unit is masked like tokens past the sequence end);
// with a page table the K/V caches are page pools and every 16-token sub-tile is placed through one table lookup,
// fetched with the index window a window of 32 units ahead (page_tokens % 16 == 0: a sub-tile never straddles pages).
#include "common.cuh"

#include <string.h>

#include <mutex>

namespace spot {

namespace {

constexpr int ATT_WARPS = 4;
constexpr int ATT_STAGES = 3;
constexpr int ATT_D = 128;
constexpr int SUB_TOK = 16;                               // tokens per warp per block
constexpr int STAGE_BYTES = 2 * SUB_TOK * ATT_D * 2;      // K + V sub-tiles: 8 KiB
constexpr int ATT_SMEM = ATT_WARPS * ATT_STAGES * STAGE_BYTES;   // 96 KiB -> 2 CTAs per SM

struct AttnArgs {
    const uint16_t* q;
    const uint16_t* k;
    const uint16_t* v;
    int64_t sb, st, sh;          // element strides: batch, token, head
    const int32_t* seq_len;
    int max_len;                 // host-side bound of seq_len: device values are clamped to [0, max_len]
    const int32_t* indices;      // nullptr: dense
    const int32_t* budgets;
    int cap;
    int fine;                    // 16-token blocks (f3): a unit is four consecutive list entries, one per warp
    const int32_t* page_table;   // nullptr: contiguous caches; else k / v are page pools (f3, R32)
    int pt_stride, page_tokens, page_vtok;   // page_vtok = page stride in units of the token stride
    int B, H_q, H_kv, G;
    float scale_log2;            // sm_scale * log2(e)
    int n_ctas;                  // gridDim.x of attn_decode_kernel (the merge kernel recomputes the same cut)
    int n_phases;                // 1, or 2 in a pipelined step with B >= 2: sequences [0, ceil(B/2)) first, then the rest
    StepSync sync;               // pipelined step: ready[b] of the selection kernel (tag == 0: stream order)
    long long phase_slots;       // partial slots per phase (>= n_ctas + B*H_kv)
    float* part_o;               // [2 * phase_slots][G][128]
    float* part_ml;              // [2 * phase_slots][G][2]
    uint16_t* out;
    float* lse;
};

__device__ __forceinline__ int seq_len_of(const AttnArgs& a, int b) { return min(max(a.seq_len[b], 0), a.max_len); }
// list entries of sequence b (sparse form)
__device__ __forceinline__ int seq_entries(const AttnArgs& a, int b) { return max(0, min(a.budgets[b], a.cap)); }
// units of sequence b per KV head: 64 tokens each -- a selected 64-token block, four selected 16-token blocks (the
// last unit of a list may be short), or a 64-token stretch of the whole sequence (dense)
__device__ __forceinline__ int seq_blocks(const AttnArgs& a, int b) {
    if (!a.indices) return (seq_len_of(a, b) + 63) >> 6;
    const int n = seq_entries(a, b);
    return a.fine ? (n + 3) >> 2 : n;
}

// A pipelined step cuts the unit list twice: sequences [0, split) first, then [split, B), split = ceil(B / 2).  The first
// half's index lists are ready when the scoring stream ends (their selection ran beside the scoring of the second half);
// the second half's are long there when a CTA finishes its first range.
// (Measured and not kept, end of round 2: phase 0 = the scoring grid's FIRST group, B / 4 sequences, whose lists are the ones
// ready when the scoring stream ends -- at B = 8, L = 32K attention then starts 5 us earlier, and the step got 5 us LONGER
// (113.9 -> 119.1 us; B = 4 and 16 unchanged): a phase of ~11 units per CTA is all ramp.)
__device__ __forceinline__ int phase_split(const AttnArgs& a) { return (a.B + 1) >> 1; }
__device__ __forceinline__ int phase_lo(const AttnArgs& a, int phase) { return (a.n_phases == 2 && phase == 1) ? phase_split(a) : 0; }
__device__ __forceinline__ int phase_hi(const AttnArgs& a, int phase) { return (a.n_phases == 2 && phase == 0) ? phase_split(a) : a.B; }

// (Measured and not kept, round 2: equal shares are not equal times -- with every SM streaming at once CTAs finish the
// same number of bytes up to 25 % apart -- so the last quarter of a phase was handed out in 4-unit chunks to whoever
// finished first.  The CTAs then ended within 5 us of each other instead of 28, but the phase itself only got 2 us
// shorter: the stream already runs at 6.4 TB/s, the HBM ceiling, and the stragglers' tail was using the bandwidth the
// finished CTAs had left; the merge kernel paid 8 us for the extra partials.)

// smem sub-tile: [16 rows][256 B], 16-byte chunk index XOR-swizzled with (row & 7)
__device__ __forceinline__ uint32_t sw_off(int row, int chunk) { return (uint32_t)(row * 256 + ((chunk ^ (row & 7)) << 4)); }

// tok0: the sub-tile's first LOGICAL token (rows at or past L are zero-filled); vtok0: where it lives, in units of
// the token stride from kbase / vbase (== tok0 unless the cache is paged)
__device__ __forceinline__ void issue_subtile(uint32_t smem_stage, const uint16_t* kbase, const uint16_t* vbase,
                                              int64_t st, int tok0, int vtok0, int L, int lane) {
    // 16 rows x 16 chunks of 16 B for K and again for V: 8 + 8 cp.async per lane
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        int id = i * 32 + lane;
        int row = id >> 4, ch = id & 15;
        bool ok = tok0 + row < L;
        int64_t off = (int64_t)(ok ? vtok0 + row : 0) * st + ch * 8;
        cp_async16(smem_stage + sw_off(row, ch), kbase + off, ok);
        cp_async16(smem_stage + SUB_TOK * 256 + sw_off(row, ch), vbase + off, ok);
    }
}

__global__ void __launch_bounds__(ATT_WARPS * 32, 2) attn_decode_kernel(AttnArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, c = lane & 3;
    const int G = a.G;
    const bool piped = a.sync.tag != 0u;
    SPOT_STAMP(a.sync, 2, 0);
#ifdef SPOT_TRACE
    if (a.sync.trace && threadIdx.x == 0 && blockIdx.x < 512) {
        unsigned sm;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
        a.sync.trace[((size_t)7 * 512 + blockIdx.x) * 4] = sm;
    }
#endif
    if (piped) {
        pdl_launch_dependents();                     // (the index lists are awaited sequence by sequence below)
    } else {
        pdl_wait();
        pdl_launch_dependents();
    }
    const uint32_t my_smem = smem_u32(smem) + warp * (ATT_STAGES * STAGE_BYTES);

  // A pipelined step runs the stream-K cut twice (phase_split above) -- so no selection latency is left between the
  // scoring stream and this one.
  for (int phase = 0; phase < a.n_phases; ++phase) {
    const int b_lo = phase_lo(a, phase), b_hi = phase_hi(a, phase);
    if (piped) {
        if (threadIdx.x == 0)
            for (int bb = b_lo; bb < b_hi; ++bb) spin_until_eq(a.sync.ready + bb, a.sync.tag);
        __syncthreads();
        SPOT_STAMP(a.sync, 2, 1 + phase);
    }
    // this CTA's range of the phase's flat unit list
    long long U = 0;
    for (int bb = b_lo; bb < b_hi; ++bb) U += seq_blocks(a, bb);
    U *= a.H_kv;
    // with fewer units than CTAs only the first U CTAs work (one unit each): every working CTA owns >= 1 unit, which
    // is what lets the merge kernel skip per-CTA emptiness checks
    const long long n_eff = U < (long long)gridDim.x ? U : (long long)gridDim.x;
    if ((long long)blockIdx.x >= n_eff) continue;
    const long long u0 = (long long)blockIdx.x * U / n_eff, u1 = (long long)(blockIdx.x + 1) * U / n_eff;
    if (u0 >= u1) continue;
    const int64_t slot0 = (int64_t)phase * a.phase_slots + blockIdx.x;      // partial slot = phase * slots + CTA + segment
    int b = b_lo, nb = seq_blocks(a, b_lo);
    long long base = 0;
    while (u0 >= base + (long long)a.H_kv * nb) { base += (long long)a.H_kv * nb; ++b; nb = seq_blocks(a, b); }
    int hk = (int)((u0 - base) / nb);
    int jbeg = (int)(u0 - base - (long long)hk * nb);

    for (long long u = u0; u < u1;) {
        const int jend = (int)min((long long)nb, (long long)jbeg + (u1 - u));
        const int n_it = jend - jbeg;
        if (n_it > 0) {
            const int L = seq_len_of(a, b);
            // Q fragments (A operand): rows = query heads of this KV group, zero-padded to 16.
            uint32_t qa[8][4];
            {
                const uint16_t* qb = a.q + ((int64_t)b * a.H_q + (int64_t)hk * G) * ATT_D;
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    int col = ks * 16 + c * 2;
                    qa[ks][0] = (g < G) ? *reinterpret_cast<const uint32_t*>(qb + g * ATT_D + col) : 0u;
                    qa[ks][1] = (g + 8 < G) ? *reinterpret_cast<const uint32_t*>(qb + (g + 8) * ATT_D + col) : 0u;
                    qa[ks][2] = (g < G) ? *reinterpret_cast<const uint32_t*>(qb + g * ATT_D + col + 8) : 0u;
                    qa[ks][3] = (g + 8 < G) ? *reinterpret_cast<const uint32_t*>(qb + (g + 8) * ATT_D + col + 8) : 0u;
                }
            }
            const bool paged = a.page_table != nullptr;
            const int64_t hbase = (paged ? 0 : (int64_t)b * a.sb) + (int64_t)hk * a.sh;
            const uint16_t* kbase = a.k + hbase;
            const uint16_t* vbase = a.v + hbase;
            const int32_t* ptab = paged ? a.page_table + (int64_t)b * a.pt_stride : nullptr;
            const bool fine = a.fine != 0;
            const int n_ent = fine ? seq_entries(a, b) : 0;
            const int32_t* idx = a.indices ? a.indices + (int64_t)b * a.cap + (fine ? 0 : jbeg) : nullptr;

            float o[16][4];
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
            float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;

            // first token of this warp's 16-token sub-tile of every unit of the portion, 32 units per window, one per
            // lane; the next window is fetched a window ahead.  (A list entry past the budget: a token past L, masked.)
            auto load_ids = [&](int w) -> int {
                const int it = w * 32 + lane;
                if (it >= n_it) return 0;
                if (fine) {
                    const int e = (jbeg + it) * 4 + warp;
                    return e < n_ent ? idx[e] * 16 : 0x3fffff00;
                }
                return (idx ? idx[it] : (jbeg + it)) * 64 + warp * SUB_TOK;
            };
            // paged: the sub-tile's place in the pool (a sub-tile never straddles a page: page_tokens % 16 == 0)
            auto place = [&](int tok) -> int {
                if (!paged || tok >= L) return tok;
                const int lp = tok / a.page_tokens;
                return ptab[lp] * a.page_vtok + (tok - lp * a.page_tokens);
            };
            int ids_cur = load_ids(0), ids_nxt = load_ids(1), win = 0;
            int vid_cur = place(ids_cur), vid_nxt = place(ids_nxt);
            auto tok_at = [&](int it) -> int {
                return __shfl_sync(0xffffffffu, (it >> 5) == win ? ids_cur : ids_nxt, it & 31);
            };
            auto vtok_at = [&](int it, int tok) -> int {
                return paged ? __shfl_sync(0xffffffffu, (it >> 5) == win ? vid_cur : vid_nxt, it & 31) : tok;
            };
            // prologue: fill STAGES-1 stages
#pragma unroll
            for (int s = 0; s < ATT_STAGES - 1; ++s) {
                if (s < n_it) {
                    const int t = tok_at(s);
                    issue_subtile(my_smem + s * STAGE_BYTES, kbase, vbase, a.st, t, vtok_at(s, t), L, lane);
                }
                cp_async_commit();
            }

            for (int it = 0; it < n_it; ++it) {
                if ((it >> 5) != win) {
                    win = it >> 5;
                    ids_cur = ids_nxt; ids_nxt = load_ids(win + 1);
                    vid_cur = vid_nxt; vid_nxt = place(ids_nxt);
                }
                {
                    int nx = it + ATT_STAGES - 1;
                    if (nx < n_it) {
                        const int t = tok_at(nx);
                        issue_subtile(my_smem + (nx % ATT_STAGES) * STAGE_BYTES, kbase, vbase, a.st, t, vtok_at(nx, t),
                                      L, lane);
                    }
                    cp_async_commit();
                }
                cp_async_wait<ATT_STAGES - 1>();
                __syncwarp();

                const uint32_t ks_base = my_smem + (it % ATT_STAGES) * STAGE_BYTES;
                const uint32_t vs_base = ks_base + SUB_TOK * 256;
                const int tok0 = tok_at(it);

                // S = Q K^T : 16 (heads) x 16 (tokens), k = 128
                float s[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
                {
                    const int mi = lane >> 3, r8 = lane & 7;
                    const int row = (mi >> 1) * 8 + r8;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        uint32_t b0, b1, b2, b3;
                        ldmatrix_x4(b0, b1, b2, b3, ks_base + sw_off(row, 2 * ks + (mi & 1)));
                        mma_bf16_16816(s[0], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b0, b1);
                        mma_bf16_16816(s[1], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b2, b3);
                    }
                }
                // scale to the log2 domain, mask tokens beyond the sequence (only a ragged last block has any)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        int tok = tok0 + nt * 8 + c * 2 + (e & 1);
                        s[nt][e] = (tok < L) ? s[nt][e] * a.scale_log2 : -INFINITY;
                    }
                // online softmax, rows g (m0, l0) and g + 8 (m1, l1)
                float mx0 = fmaxf(fmaxf(s[0][0], s[0][1]), fmaxf(s[1][0], s[1][1]));
                float mx1 = fmaxf(fmaxf(s[0][2], s[0][3]), fmaxf(s[1][2], s[1][3]));
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
                for (int nt = 0; nt < 2; ++nt) {
                    s[nt][0] = fast_exp2(s[nt][0] - mu0); s[nt][1] = fast_exp2(s[nt][1] - mu0);
                    s[nt][2] = fast_exp2(s[nt][2] - mu1); s[nt][3] = fast_exp2(s[nt][3] - mu1);
                    ps0 += s[nt][0] + s[nt][1];
                    ps1 += s[nt][2] + s[nt][3];
                }
                l0 = l0 * c0 + ps0;
                l1 = l1 * c1 + ps1;
#pragma unroll
                for (int i = 0; i < 16; ++i) { o[i][0] *= c0; o[i][1] *= c0; o[i][2] *= c1; o[i][3] *= c1; }

                // O += P V : P (16 x 16 tokens) as A, V (16 tokens x 128) as B through ldmatrix.trans
                const uint32_t pa0 = pack_bf16x2(s[0][0], s[0][1]), pa1 = pack_bf16x2(s[0][2], s[0][3]);
                const uint32_t pa2 = pack_bf16x2(s[1][0], s[1][1]), pa3 = pack_bf16x2(s[1][2], s[1][3]);
                {
                    const int mi = lane >> 3, r8 = lane & 7;
                    const int row = (mi & 1) * 8 + r8;
#pragma unroll
                    for (int nd = 0; nd < 16; nd += 2) {
                        uint32_t b0, b1, b2, b3;
                        ldmatrix_x4_trans(b0, b1, b2, b3, vs_base + sw_off(row, nd + (mi >> 1)));
                        mma_bf16_16816(o[nd], pa0, pa1, pa2, pa3, b0, b1);
                        mma_bf16_16816(o[nd + 1], pa0, pa1, pa2, pa3, b2, b3);
                    }
                }
                __syncwarp();   // everyone is done reading this stage before a later iteration refills it
            }
            cp_async_wait<0>();

            // full row sums
            l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
            l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);

            // merge the 4 warps through shared memory (the rings are idle now)
            __syncthreads();
            float* so = reinterpret_cast<float*>(smem);                  // [warp][16][128]
            float* sml = so + ATT_WARPS * 16 * ATT_D;                    // [warp][16][2]
#pragma unroll
            for (int nd = 0; nd < 16; ++nd) {
                int col = nd * 8 + c * 2;
                *reinterpret_cast<float2*>(so + (warp * 16 + g) * ATT_D + col) = make_float2(o[nd][0], o[nd][1]);
                *reinterpret_cast<float2*>(so + (warp * 16 + g + 8) * ATT_D + col) = make_float2(o[nd][2], o[nd][3]);
            }
            if (c == 0) {
                sml[(warp * 16 + g) * 2] = m0; sml[(warp * 16 + g) * 2 + 1] = l0;
                sml[(warp * 16 + g + 8) * 2] = m1; sml[(warp * 16 + g + 8) * 2 + 1] = l1;
            }
            __syncthreads();
            const int64_t pbase = (slot0 + (int64_t)b * a.H_kv + hk) * G;
            for (int r = 0; r < G; ++r) {
                float mw[ATT_WARPS], M = -INFINITY;
#pragma unroll
                for (int w = 0; w < ATT_WARPS; ++w) { mw[w] = sml[(w * 16 + r) * 2]; M = fmaxf(M, mw[w]); }
                const float Mu = (M == -INFINITY) ? 0.f : M;
                float acc = 0.f, lsum = 0.f;
#pragma unroll
                for (int w = 0; w < ATT_WARPS; ++w) {
                    float f = fast_exp2(mw[w] - Mu);
                    acc += f * so[(w * 16 + r) * ATT_D + threadIdx.x];
                    lsum += f * sml[(w * 16 + r) * 2 + 1];
                }
                a.part_o[(pbase + r) * ATT_D + threadIdx.x] = acc;
                if (threadIdx.x == 0) { a.part_ml[(pbase + r) * 2] = M; a.part_ml[(pbase + r) * 2 + 1] = lsum; }
            }
            __syncthreads();    // the rings are reused by the next portion
        }
        u += n_it;
        jbeg = jend;
        if (jbeg >= nb) {
            jbeg = 0;
            if (++hk == a.H_kv) { hk = 0; ++b; nb = (b < b_hi) ? seq_blocks(a, b) : 1; }
        }
    }
  }
    SPOT_STAMP(a.sync, 2, 3);
    if (piped && threadIdx.x == 0) pdl_wait();      // completion of this grid implies completion of its predecessors
}

// merge the partials of one (sequence, query head): one warp each.  The contributors of segment s = (b, hk) are the
// CTAs whose ranges overlap the segment's units; their slots are CTA + s.
constexpr int MERGE_WARPS = 8;
__global__ void __launch_bounds__(MERGE_WARPS * 32) attn_merge_kernel(AttnArgs a) {
    // one CTA per (sequence, query head); its warps split the row's partials between them
    __shared__ float s_acc[MERGE_WARPS][ATT_D + 4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int row = blockIdx.x;
    SPOT_STAMP(a.sync, 3, 0);
    const int b = row / a.H_q, h = row - b * a.H_q;
    const int G = a.G, hk = h / G, r = h - hk * G;
    // In a pipelined step this kernel is resident long before the attention grid completes, and its code comes from DRAM
    // (the bench flushes L2 before every step): a cold pass costs several us at the very end of the step.  So the body
    // runs once DRY before griddepcontrol.wait -- on slot 0 of the workspace, nothing stored -- and then for real.
#pragma unroll 1
    for (int pass = a.sync.tag ? 0 : 1; pass < 2; ++pass) {
        const bool dry = pass == 0;
        // contributors: the CTAs c_first .. c_last whose ranges overlap the segment
        int c_first = 0, c_last = 0, nb = 1;
        int64_t base_slot = 0;               // + CTA: the contributor's partial slot of this segment
        if (!dry) {
            pdl_wait();
            pdl_launch_dependents();
            SPOT_STAMP(a.sync, 3, 1);
            // the attention grid has completed: nobody waits on the ready words of this call any more (common.cuh, StepSync)
            if (a.sync.tag && blockIdx.x == 0 && threadIdx.x < a.B) a.sync.ready[threadIdx.x] = 0u;
            // the phase that covered this sequence
            const int phase = (a.n_phases == 2 && b >= phase_split(a)) ? 1 : 0;
            const int b_lo = phase_lo(a, phase), b_hi = phase_hi(a, phase);
            long long U = 0, before = 0;
            for (int bb = b_lo; bb < b_hi; ++bb) {
                const int n = seq_blocks(a, bb);
                if (bb < b) before += n;
                U += n;
            }
            U *= a.H_kv;
            nb = seq_blocks(a, b);
            if (nb > 0) {
                const long long us = before * a.H_kv + (long long)hk * nb, ue = us + nb;
                const long long n = U < (long long)a.n_ctas ? U : (long long)a.n_ctas;     // working CTAs (same rule as the kernel)
                c_first = (int)(((us + 1) * n - 1) / U);
                c_last = (int)((ue * n - 1) / U);
                base_slot = (int64_t)phase * a.phase_slots + (int64_t)b * a.H_kv + hk;
            }
        }
        const int n_contrib = c_last - c_first + 1;
        auto slot_of = [&](int t) -> int64_t { return base_slot + c_first + t; };
        uint16_t* outp = a.out + ((int64_t)b * a.H_q + h) * ATT_D + lane * 4;
        if (nb == 0) {                       // (block-uniform) an empty list: zeros, LSE = -inf
            if (warp == 0) {
                *reinterpret_cast<uint2*>(outp) = make_uint2(0u, 0u);
                if (a.lse && lane == 0) a.lse[(int64_t)b * a.H_q + h] = -INFINITY;
            }
            return;
        }
        // Every warp folds its share of the contributors with a running maximum of its own (online log-sum-exp: no pass over
        // all the maxima in front of the loads -- one L2 round trip less on the tail of the step), four partials in flight
        // at a time; warp 0 then combines the warps' (m, l, acc).
        float m_w = -INFINITY, lsum = 0.f;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int t0 = warp; t0 < n_contrib; t0 += 4 * MERGE_WARPS) {
            float2 ml[4];
            float4 o[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int t = t0 + u * MERGE_WARPS;
                ml[u] = make_float2(-INFINITY, 0.f);
                o[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (t < n_contrib) {
                    const int64_t pr = slot_of(t) * G + r;
                    ml[u] = *reinterpret_cast<const float2*>(a.part_ml + pr * 2);
                    o[u] = *reinterpret_cast<const float4*>(a.part_o + pr * ATT_D + lane * 4);
                }
            }
            float m_new = m_w;
#pragma unroll
            for (int u = 0; u < 4; ++u) m_new = fmaxf(m_new, ml[u].x);
            if (m_new > -INFINITY) {
                const float f_old = fast_exp2(m_w - m_new);        // exp2(-inf) = 0 on the first contributors
                acc.x *= f_old; acc.y *= f_old; acc.z *= f_old; acc.w *= f_old;
                lsum *= f_old;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float f = fast_exp2(ml[u].x - m_new);    // (a padding entry has m = -inf: f = 0)
                    acc.x += f * o[u].x; acc.y += f * o[u].y; acc.z += f * o[u].z; acc.w += f * o[u].w;
                    lsum += f * ml[u].y;
                }
                m_w = m_new;
            }
        }
        *reinterpret_cast<float4*>(&s_acc[warp][lane * 4]) = acc;
        if (lane == 0) { s_acc[warp][ATT_D] = lsum; s_acc[warp][ATT_D + 1] = m_w; }
        __syncthreads();
        if (warp == 0) {
            float M = -INFINITY;
#pragma unroll
            for (int w = 0; w < MERGE_WARPS; ++w) M = fmaxf(M, s_acc[w][ATT_D + 1]);
            const float Mu = (M == -INFINITY) ? 0.f : M;
            acc = make_float4(0.f, 0.f, 0.f, 0.f);
            lsum = 0.f;
#pragma unroll
            for (int w = 0; w < MERGE_WARPS; ++w) {
                const float f = fast_exp2(s_acc[w][ATT_D + 1] - Mu);
                const float4 o = *reinterpret_cast<const float4*>(&s_acc[w][lane * 4]);
                acc.x += f * o.x; acc.y += f * o.y; acc.z += f * o.z; acc.w += f * o.w;
                lsum += f * s_acc[w][ATT_D];
            }
            const float inv = lsum > 0.f ? 1.f / lsum : 0.f;
            if (!dry) {
                *reinterpret_cast<uint2*>(outp) =
                    make_uint2(pack_bf16x2(acc.x * inv, acc.y * inv), pack_bf16x2(acc.z * inv, acc.w * inv));
                if (a.lse && lane == 0)
                    a.lse[(int64_t)b * a.H_q + h] = (lsum > 0.f) ? (M + log2f(lsum)) * 0.6931471805599453f : -INFINITY;
            }
        }
        __syncthreads();                     // s_acc is reused by the next pass
    }
    SPOT_STAMP(a.sync, 3, 2);
}

// persistent grid: two CTAs per SM, never more CTAs than units
int pick_ctas(const spot_attn_params* p, bool dense) {
    int64_t max_blocks = dense ? (p->max_seq_len + 63) / 64 : p->cap;
    int64_t units = max_blocks * p->H_kv * p->B;
    int64_t want = (int64_t)sm_count() * 2;
    return (int)(units < want ? (units < 1 ? 1 : units) : want);
}

spot_status check_attn(const spot_attn_params* p, bool dense, bool prefill) {
    if (!p || !p->q || !p->k || !p->v || !p->out) return SPOT_ERR_INVALID_ARG;
    if (!aligned16(p->q) || !aligned16(p->k) || !aligned16(p->v) || !aligned16(p->out)) return SPOT_ERR_INVALID_ARG;
    if (p->B <= 0 || p->H_q <= 0 || p->H_kv <= 0 || p->H_q % p->H_kv != 0) return SPOT_ERR_INVALID_ARG;
    if (p->H_q / p->H_kv > 16) return SPOT_ERR_UNSUPPORTED;
    if (p->D != 128 || (p->blk != 64 && !(p->blk == 16 && !prefill))) return SPOT_ERR_UNSUPPORTED;
    if (p->kv_stride_token < p->D || p->kv_stride_token % 8 || p->kv_stride_head % 8 || p->kv_stride_batch % 8)
        return SPOT_ERR_INVALID_ARG;
    if (!dense && p->indices && (!p->budgets || p->cap <= 0)) return SPOT_ERR_INVALID_ARG;
    if (!prefill) {
        if (!p->seq_len || p->max_seq_len <= 0) return SPOT_ERR_INVALID_ARG;
    }
    if (p->page_table) {
        if (prefill) return SPOT_ERR_UNSUPPORTED;
        if (p->page_tokens <= 0 || p->page_tokens % 16 != 0) return SPOT_ERR_INVALID_ARG;
        if ((int64_t)p->page_table_stride * p->page_tokens < p->max_seq_len) return SPOT_ERR_INVALID_ARG;
        if (p->kv_stride_batch <= 0 || p->kv_stride_batch % p->kv_stride_token != 0) return SPOT_ERR_INVALID_ARG;
    }
    return SPOT_OK;
}

// partial slots of one phase: CTA + segment; sized for the two phases of a pipelined step whether or not the call is one
int64_t phase_slot_count(const spot_attn_params* p, bool dense) {
    const bool use_idx = !dense && p->indices;
    return (int64_t)pick_ctas(p, !use_idx) + (int64_t)p->B * p->H_kv;
}
size_t decode_ws_bytes(const spot_attn_params* p, bool dense) {
    return (size_t)(2 * phase_slot_count(p, dense) * (p->H_q / p->H_kv) * (ATT_D + 2) * 4);
}

// sync: the hand-offs of a pipelined step (spot_decode_step; nullptr: plain stream order).  In a step the grid leaves
// out the SMs that the selection CTAs of the second half of the batch may still hold when the attention CTAs become
// resident: a CTA that starts late would finish its (equal) share late.
spot_status run_decode(const spot_attn_params* p, bool dense, const StepSync* sync, cudaStream_t s) {
    spot_status stt = check_attn(p, dense, false);
    if (stt != SPOT_OK) return stt;
    if ((stt = check_device()) != SPOT_OK) return stt;
    const bool use_idx = !dense && p->indices;
    int n_ctas = pick_ctas(p, !use_idx);
    const int G = p->H_q / p->H_kv;
    const int64_t phase_slots = phase_slot_count(p, dense);
    const int64_t slots = 2 * phase_slots;
    const size_t need = (size_t)(slots * G * (ATT_D + 2) * 4);
    if (!p->workspace || p->workspace_bytes < need) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    AttnArgs a;
    memset(&a.sync, 0, sizeof(a.sync));
    a.n_phases = 1;
    a.phase_slots = phase_slots;
    if (sync && use_idx) {
        a.sync = *sync;
        if (p->B >= 2) {
            a.n_phases = 2;
            const int second_half = p->B - (p->B + 1) / 2;
            const int fewer = 2 * (sm_count() - (second_half < 8 ? second_half : 8));
            if (n_ctas > fewer && fewer > 0) n_ctas = fewer;
        }
    }
    a.q = p->q; a.k = p->k; a.v = p->v;
    a.sb = p->kv_stride_batch; a.st = p->kv_stride_token; a.sh = p->kv_stride_head;
    a.seq_len = p->seq_len; a.max_len = p->max_seq_len; a.indices = use_idx ? p->indices : nullptr; a.budgets = p->budgets; a.cap = p->cap;
    a.fine = use_idx && p->blk == 16;
    a.page_table = p->page_table; a.pt_stride = p->page_table_stride; a.page_tokens = p->page_tokens;
    a.page_vtok = p->page_table ? (int)(p->kv_stride_batch / p->kv_stride_token) : 0;
    a.B = p->B; a.H_q = p->H_q; a.H_kv = p->H_kv; a.G = G;
    a.scale_log2 = p->sm_scale * 1.4426950408889634f;
    a.n_ctas = n_ctas;
    a.part_o = reinterpret_cast<float*>(p->workspace);
    a.part_ml = a.part_o + slots * G * ATT_D;
    a.out = p->out; a.lse = p->lse;
    static unsigned long long smem_attr_done = 0;
    SPOT_CUDA_TRY(set_max_smem_once(attn_decode_kernel, ATT_SMEM, smem_attr_done));
    SPOT_CUDA_TRY(launch_pdl(attn_decode_kernel, dim3((unsigned)n_ctas), dim3(ATT_WARPS * 32), ATT_SMEM, s, a));
    const int rows = p->B * p->H_q;
    SPOT_CUDA_TRY(launch_pdl(attn_merge_kernel, dim3((unsigned)rows), dim3(MERGE_WARPS * 32), 0, s, a));
    return SPOT_OK;
}

}  // namespace

// ---- spot_sparse_attn_decode_static: the same call with its scratch inside the library (include/spot.h) -----------------
// The split-KV partials of attn_decode_kernel / attn_merge_kernel live in this file-scope array instead of a caller's
// workspace: nothing is allocated by the call.  Every GPU that loads the library holds the array until the process exits.
// In host code `g_static_scratch` is only a stand-in for the symbol, NOT a device address: the address comes from
// cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[SPOT_STATIC_SCRATCH_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
spot_status static_scratch_ptr(void** out) {
    static std::mutex mu;
    static void* ptr_of_device[STATIC_MAX_DEVICES] = {};
    int dev = -1;
    SPOT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return SPOT_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of_device[dev]) {
        void* ptr = nullptr;
        SPOT_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_scratch));
        if (!ptr) return SPOT_ERR_CUDA;
        ptr_of_device[dev] = ptr;
    }
    *out = ptr_of_device[dev];
    return SPOT_OK;
}

spot_status run_decode_static(const spot_attn_params* p, cudaStream_t s) {
    spot_status st = check_attn(p, false, false);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    // beyond the built-in maximum: refuse before anything is launched (the caller falls back to spot_sparse_attn_decode
    // with a workspace of its own)
    if (decode_ws_bytes(p, false) > (size_t)SPOT_STATIC_SCRATCH_BYTES) return SPOT_ERR_WORKSPACE_TOO_SMALL;
    spot_attn_params q = *p;
    void* scratch = nullptr;
    if ((st = static_scratch_ptr(&scratch)) != SPOT_OK) return st;
    q.workspace = scratch;
    q.workspace_bytes = (size_t)SPOT_STATIC_SCRATCH_BYTES;
    // Nothing in the array has to start at zero: the attention kernel writes every partial slot (o, m, l) the merge kernel
    // reads, so the previous call's contents are simply overwritten.
    return run_decode(&q, false, nullptr, s);
}

spot_status check_attn_decode_args(const spot_attn_params* p) { return check_attn(p, false, false); }
spot_status attn_decode_piped(const spot_attn_params* p, const StepSync* sync, cudaStream_t s) {
    return run_decode(p, false, sync, s);
}

}  // namespace spot

using namespace spot;

extern "C" size_t spot_sparse_attn_decode_workspace_bytes(const spot_attn_params* p) {
    if (!p || check_attn(p, false, false) != SPOT_OK) return 0;
    return decode_ws_bytes(p, false);
}
extern "C" spot_status spot_sparse_attn_decode(const spot_attn_params* p, void* stream) {
    return run_decode(p, false, nullptr, (cudaStream_t)stream);
}
extern "C" spot_status spot_sparse_attn_decode_static(const spot_attn_params* p, void* stream) {
    return run_decode_static(p, (cudaStream_t)stream);
}
extern "C" size_t spot_dense_attn_decode_workspace_bytes(const spot_attn_params* p) {
    if (!p || check_attn(p, true, false) != SPOT_OK) return 0;
    return decode_ws_bytes(p, true);
}
extern "C" spot_status spot_dense_attn_decode(const spot_attn_params* p, void* stream) {
    return run_decode(p, true, nullptr, (cudaStream_t)stream);
}
