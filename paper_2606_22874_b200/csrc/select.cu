// Step a2 -- block distribution and selection rule, one CTA per selection row:
// reserved sink/recency tier, residual softmax (Eq. 7), nucleus + K_min floor (Eq. 8) or static top-K (Eq. 6).
//
// Latency-bound (<= 8192 scores per row, 4..16 rows at decode), so the kernel is built around the critical path:
//   * every thread keeps 8 scores in registers as 32-bit order-preserving keys; element e lives at
//     (warp w, register r, lane l) with e = 256 w + 32 r + l;
//   * a bitonic sort of the KEYS ONLY (no payload): strides 1..16 are warp shuffles, strides 32..128 are
//     register-to-register, strides >= 256 go through shared memory three at a time (a transposed layout makes
//     three consecutive strides thread-local), i.e. 2 CTA barriers per three cross-warp strides instead of one per
//     stride;
//   * the mass of a block is a function of its score, so the sorted keys alone give the sorted masses: exp,
//     normalisation and the prefix mass run in fp64 on the sorted keys (the only source of disagreement with the
//     fp64 oracle is then the fp32 block score itself);
//   * the cut is a key value tau = key of rank n_take-1; blocks with a better key are selected, blocks tied with tau
//     are taken in ascending block index until n_take is reached -- exactly the (score descending, index
//     ascending) order R7 fixes -- and the ascending index list falls out of one ballot/popc scan in index order.
#include "select_common.cuh"

namespace spot {

namespace {

__device__ __forceinline__ void cmpx(uint32_t& a, uint32_t& b, bool asc) {
    const uint32_t lo = min(a, b), hi = max(a, b);
    a = asc ? lo : hi;
    b = asc ? hi : lo;
}

// LT = log2(threads); the CTA sorts NPAD = 8 << LT keys.
template <int LT>
__global__ void __launch_bounds__(1 << LT) select_kernel(SelectArgs a) {
    constexpr int T = 1 << LT;
    constexpr int NPAD = 8 * T;
    constexpr int LOGN = LT + 3;
    constexpr int NSEG = T / 4;                 // 32-element rank segments: (warp, register)
    static_assert(LT == 5 || LT >= 8, "cross-warp rounds need three register bits above bit 8");
    __shared__ uint32_t s_key[NPAD];
    __shared__ double s_seg[NSEG];
    __shared__ int s_cnt[NSEG][2];
    __shared__ double s_total;
    __shared__ uint32_t s_bcast[2];
    __shared__ int s_below;
    __shared__ int s_tot[2];

    const int row = blockIdx.x;
    const int b = row / a.n_q, i = row - b * a.n_q;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_wait();
    pdl_launch_dependents();
    int n_b;
    if (a.q_block == 1) n_b = (a.seq_len[b] + a.blk - 1) / a.blk;
    else n_b = (a.q_start + (i + 1) * a.q_block - 1) / a.blk + 1;
    n_b = min(n_b, NPAD);
    const int sink_end = min(a.sink, n_b);
    const int rec_beg = max(sink_end, n_b - a.rec);     // residual blocks: [sink_end, rec_beg)
    const int n_res = rec_beg - sink_end;
    const int n_reserved = n_b - n_res;
    const int ebase = warp * 256 + lane;                // element of register r: ebase + 32 r

    // ---- load: block scores -> keys (pads and reserved blocks sort last)
    const float* srow = a.scores + (int64_t)row * a.nb_stride;
    uint32_t okey[8], key[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int j = ebase + 32 * r;
        okey[r] = (j >= sink_end && j < rec_beg) ? score_key(srow[j]) : KEY_PAD;
        key[r] = okey[r];
    }
    if (tid == 0) { s_below = 0; }

    // ---- bitonic sort, ascending
#pragma unroll
    for (int lk = 1; lk <= LOGN; ++lk) {
        const int k = 1 << lk;
#pragma unroll
        for (int lj = lk - 1; lj >= 0; --lj) {
            if (lj >= 8) {
                // cross-warp strides, three at a time: the group whose lowest stride bit is ls is thread-local in
                // the transposed layout idx_m = low + (m << ls) + (high << (ls + 3)).
                if ((lk - 1 - lj) % 3 == 0) {            // first stride of its group: run the whole group here
                    const int cnt = (lj - 7) >= 3 ? 3 : (lj - 7);
                    const int ls = lj - cnt + 1;
#pragma unroll
                    for (int r = 0; r < 8; ++r) s_key[ebase + 32 * r] = key[r];
                    __syncthreads();
                    const int low = tid & ((1 << ls) - 1), high = tid >> ls;
                    const int tbase = low + (high << (ls + 3));
                    uint32_t v[8];
#pragma unroll
                    for (int m = 0; m < 8; ++m) v[m] = s_key[tbase + (m << ls)];
#pragma unroll
                    for (int bit = cnt - 1; bit >= 0; --bit) {
#pragma unroll
                        for (int m = 0; m < 8; ++m) {
                            // the direction bit lk may itself be a register bit (lk < ls + 3): test it per element
                            if ((m & (1 << bit)) == 0)
                                cmpx(v[m], v[m | (1 << bit)], ((tbase + (m << ls)) & k) == 0);
                        }
                    }
#pragma unroll
                    for (int m = 0; m < 8; ++m) s_key[tbase + (m << ls)] = v[m];
                    __syncthreads();
#pragma unroll
                    for (int r = 0; r < 8; ++r) key[r] = s_key[ebase + 32 * r];
                }
            } else if (lj >= 5) {
                const int rr = 1 << (lj - 5);
#pragma unroll
                for (int r = 0; r < 8; ++r)
                    if ((r & rr) == 0) cmpx(key[r], key[r | rr], ((ebase + 32 * r) & k) == 0);
            } else {
                const int j = 1 << lj;
                const bool lower = (lane & j) == 0;
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const uint32_t other = __shfl_xor_sync(0xffffffffu, key[r], j);
                    const bool asc = ((ebase + 32 * r) & k) == 0;
                    key[r] = (asc == lower) ? min(key[r], other) : max(key[r], other);
                }
            }
        }
    }
    // key[r] now holds rank ebase + 32 r of the residual blocks (ranks >= n_res are pads).

    int n_take = 0;
    double inv_total = 0.0, zmax = 0.0;
    if (a.mode == SPOT_MODE_TOPK) {
        n_take = min(max(0, a.top_k - n_reserved), n_res);
    } else {
        // Eq. 7 in fp64 on the sorted keys: z = s_bar / T, m = z of rank 0, e = exp(z - m).
        if (tid == 0) s_bcast[0] = key[0];
        __syncthreads();
        zmax = (double)key_score(s_bcast[0]) / a.temperature;
        double inc[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int rank = ebase + 32 * r;
            double e = 0.0;
            if (rank < n_res) e = exp((double)key_score(key[r]) / a.temperature - zmax);
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const double t = __shfl_up_sync(0xffffffffu, e, o);
                if (lane >= o) e += t;
            }
            inc[r] = e;                                   // inclusive prefix inside the segment
            if (lane == 31) s_seg[warp * 8 + r] = e;
        }
        __syncthreads();
        if (warp == 0) {
            // exclusive scan of the NSEG segment totals (rank order = segment order)
            constexpr int PER = (NSEG + 31) / 32;
            double v[PER], run = 0.0;
#pragma unroll
            for (int u = 0; u < PER; ++u) {
                const int s = lane * PER + u;
                v[u] = (s < NSEG) ? s_seg[s] : 0.0;
                run += v[u];
            }
            double incl = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const double t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            double off = incl - run;
#pragma unroll
            for (int u = 0; u < PER; ++u) {
                const int s = lane * PER + u;
                if (s < NSEG) s_seg[s] = off;
                off += v[u];
            }
            if (lane == 31) s_total = incl;
        }
        __syncthreads();
        const double total = s_total;
        inv_total = total > 0.0 ? 1.0 / total : 0.0;
        int below = 0;                                    // ranks whose cumulative mass is still < p
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int rank = ebase + 32 * r;
            const double cum = (s_seg[warp * 8 + r] + inc[r]) * inv_total;
            if (rank < n_res && cum < a.p) ++below;
        }
        below = __reduce_add_sync(0xffffffffu, below);
        if (lane == 0 && below) atomicAdd(&s_below, below);
        __syncthreads();
        int n_star;
        if (n_res == 0) n_star = 0;
        else if (a.p >= 1.0) n_star = n_res;
        else n_star = min(n_res, s_below + 1);
        n_take = n_star;
        const int target = min(a.kmin, n_b);
        if (n_reserved + n_take < target) n_take = min(n_res, target - n_reserved);
    }

    // ---- the cut as a key value
    if (n_take > 0) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
            if (ebase + 32 * r == n_take - 1) s_bcast[1] = key[r];
    }
    __syncthreads();
    const uint32_t tau = n_take > 0 ? s_bcast[1] : 0u;

    // ---- index order: A = reserved or strictly better than tau (certainly selected), Tt = tied with tau
    int prefA[8], prefT[8];
    uint32_t isA = 0, isT = 0;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int j = ebase + 32 * r;
        const bool resid = j >= sink_end && j < rec_beg;
        const bool fa = (j < n_b && !resid) || (resid && n_take > 0 && okey[r] < tau);
        const bool ft = resid && n_take > 0 && okey[r] == tau;
        const uint32_t ba = __ballot_sync(0xffffffffu, fa), bt = __ballot_sync(0xffffffffu, ft);
        const uint32_t lt = (1u << lane) - 1u;
        prefA[r] = __popc(ba & lt);
        prefT[r] = __popc(bt & lt);
        isA |= (uint32_t)fa << r;
        isT |= (uint32_t)ft << r;
        if (lane == 0) { s_cnt[warp * 8 + r][0] = __popc(ba); s_cnt[warp * 8 + r][1] = __popc(bt); }
    }
    __syncthreads();
    if (warp == 0) {
        constexpr int PER = (NSEG + 31) / 32;
        int va[PER], vt[PER], ra = 0, rt = 0;
#pragma unroll
        for (int u = 0; u < PER; ++u) {
            const int s = lane * PER + u;
            va[u] = (s < NSEG) ? s_cnt[s][0] : 0;
            vt[u] = (s < NSEG) ? s_cnt[s][1] : 0;
            ra += va[u]; rt += vt[u];
        }
        int ia = ra, it = rt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int ta = __shfl_up_sync(0xffffffffu, ia, o), tt = __shfl_up_sync(0xffffffffu, it, o);
            if (lane >= o) { ia += ta; it += tt; }
        }
        int oa = ia - ra, ot = it - rt;
#pragma unroll
        for (int u = 0; u < PER; ++u) {
            const int s = lane * PER + u;
            if (s < NSEG) { s_cnt[s][0] = oa; s_cnt[s][1] = ot; }
            oa += va[u]; ot += vt[u];
        }
        if (lane == 31) { s_tot[0] = ia; s_tot[1] = it; }
    }
    __syncthreads();
    const int total_A = s_tot[0], total_T = s_tot[1];
    const int need = n_take - (total_A - n_reserved);    // ties to take, lowest block index first
    const int total_sel = total_A + min(total_T, max(need, 0));
    int32_t* out = a.indices + (int64_t)row * a.cap;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int j = ebase + 32 * r;
        const int a_before = s_cnt[warp * 8 + r][0] + prefA[r];
        const int t_before = s_cnt[warp * 8 + r][1] + prefT[r];
        int pos = -1;
        if ((isA >> r) & 1u) pos = a_before + min(t_before, need);
        else if (((isT >> r) & 1u) && t_before < need) pos = a_before + t_before;
        if (pos >= 0 && pos < a.cap) out[pos] = j;
    }
    for (int j = total_sel + tid; j < a.cap; j += T) out[j] = -1;
    if (tid == 0) a.budgets[row] = min(total_sel, a.cap);

    if (a.probs) {
        float* pr = a.probs + (int64_t)row * a.nb_stride;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int j = ebase + 32 * r;
            if (j < n_b) {
                float pv = 0.f;
                if (a.mode != SPOT_MODE_TOPK && j >= sink_end && j < rec_beg)
                    pv = (float)(exp((double)key_score(okey[r]) / a.temperature - zmax) * inv_total);
                pr[j] = pv;
            }
        }
    }
}

template <int LT>
spot_status launch_select(const SelectArgs& a, int rows, cudaStream_t s) {
    SPOT_CUDA_TRY(launch_pdl(select_kernel<LT>, dim3((unsigned)rows), dim3(1 << LT), 0, s, a));
    return SPOT_OK;
}

}  // namespace

spot_status launch_select_hist(const SelectArgs& a, int rows, cudaStream_t s);    // select_hist.cu

spot_status run_select(const spot_select_params* p, const float* scores, int nb_stride, int rows_per_seq,
                       int max_nb, cudaStream_t s) {
    if (max_nb > SEL_MAX_NB) return SPOT_ERR_UNSUPPORTED;
    SelectArgs a;
    a.scores = scores; a.nb_stride = nb_stride; a.seq_len = p->seq_len; a.n_q = rows_per_seq;
    a.q_start = p->q_start; a.q_block = p->q_block; a.blk = p->blk;
    a.mode = p->mode; a.top_k = p->top_k; a.p = p->p; a.temperature = p->temperature;
    a.sink = p->sink_blocks; a.rec = p->recency_blocks; a.kmin = p->kmin_blocks;
    a.indices = p->indices; a.cap = p->cap; a.budgets = p->budgets; a.probs = p->block_probs;
    const int rows = p->B * rows_per_seq;
    if (max_nb <= 2048) return launch_select_hist(a, rows, s);     // histogram-partition form
    if (max_nb <= 4096) return launch_select<9>(a, rows, s);
    return launch_select<10>(a, rows, s);
}

}  // namespace spot
