// Step a2 -- block distribution and selection rule, one CTA per selection row:
// reserved sink/recency tier, residual softmax (Eq. 7), nucleus + K_min floor (Eq. 8) or static top-K (Eq. 6).
//
// Latency-bound (<= 8192 scores per row).  The residual blocks are sorted in shared memory by the 64-bit key
// (~orderable(score), block id) -- ascending key order is (score descending, index ascending), the order R7 fixes.
// The mass arithmetic (exp, normalisation, prefix sum, threshold test) runs in fp64 so that the only source of
// disagreement with the fp64 oracle is the fp32 block score itself.
#include "common.cuh"

namespace spot {

namespace {

constexpr int SEL_THREADS = 1024;
constexpr int SEL_MAX_NB = 8192;

__device__ __forceinline__ uint32_t orderable(float x) {
    uint32_t u = __float_as_uint(x + 0.0f);   // -0.0 -> +0.0
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float from_orderable(uint32_t o) {
    uint32_t u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
    return __uint_as_float(u);
}

// inclusive scan of one double per thread across the CTA; `warp_tot` is a 32-entry shared scratch.
__device__ double block_inclusive_scan(double v, double* warp_tot, double* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        double t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    __syncthreads();
    if (lane == 31) warp_tot[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double t = warp_tot[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            double u = __shfl_up_sync(0xffffffffu, t, o);
            if (lane >= o) t += u;
        }
        warp_tot[lane] = t;
    }
    __syncthreads();
    double off = warp ? warp_tot[warp - 1] : 0.0;
    *total = warp_tot[31];
    return v + off;
}

__device__ int block_inclusive_scan_int(int v, int* warp_tot, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    __syncthreads();
    if (lane == 31) warp_tot[warp] = v;
    __syncthreads();
    if (warp == 0) {
        int t = warp_tot[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int u = __shfl_up_sync(0xffffffffu, t, o);
            if (lane >= o) t += u;
        }
        warp_tot[lane] = t;
    }
    __syncthreads();
    int off = warp ? warp_tot[warp - 1] : 0;
    *total = warp_tot[31];
    return v + off;
}

struct SelectArgs {
    const float* scores;      // [rows][nb_stride]
    int nb_stride;
    const int32_t* seq_len;   // decode: [B]; prefill: nullptr
    int n_q;                  // rows per sequence
    int q_start, q_block, blk;
    int mode, top_k;
    double p, temperature;
    int sink, rec, kmin;
    int32_t* indices;
    int cap;
    int32_t* budgets;
    float* probs;             // optional [rows][nb_stride]
};

__global__ void __launch_bounds__(SEL_THREADS) select_kernel(SelectArgs a, int n_pow2_max) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* key = reinterpret_cast<uint64_t*>(smem_raw);                      // [n_pow2]
    double* mass = reinterpret_cast<double*>(smem_raw + (size_t)n_pow2_max * 8);   // [n_pow2]
    uint8_t* flag = reinterpret_cast<uint8_t*>(smem_raw + (size_t)n_pow2_max * 16); // [n_pow2]
    __shared__ double wtot[32];
    __shared__ int itot[32];
    __shared__ int s_nstar;

    const int row = blockIdx.x;
    const int b = row / a.n_q, i = row - b * a.n_q;
    const int tid = threadIdx.x;
    int n_b;
    if (a.q_block == 1) n_b = (a.seq_len[b] + a.blk - 1) / a.blk;
    else n_b = (a.q_start + (i + 1) * a.q_block - 1) / a.blk + 1;
    n_b = min(n_b, SEL_MAX_NB);
    const int sink_end = min(a.sink, n_b);
    const int rec_beg = max(0, n_b - a.rec);
    int n_reserved = sink_end + (n_b - max(rec_beg, sink_end));
    const int n_res = n_b - n_reserved;
    int n = 1;
    while (n < n_b) n <<= 1;

    const float* srow = a.scores + (int64_t)row * a.nb_stride;
    for (int j = tid; j < n; j += SEL_THREADS) {
        uint64_t k = ~0ull;
        if (j < n_b && j >= sink_end && j < rec_beg) k = ((uint64_t)(~orderable(srow[j])) << 32) | (uint32_t)j;
        key[j] = k;
        flag[j] = (j < n_b && !(j >= sink_end && j < rec_beg)) ? 1 : 0;
    }
    if (tid == 0) s_nstar = 0;
    __syncthreads();

    // bitonic sort, ascending
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = tid; t < (n >> 1); t += SEL_THREADS) {
                int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                int hi = lo | j;
                bool asc = (lo & k) == 0;
                uint64_t x = key[lo], y = key[hi];
                if ((x > y) == asc) { key[lo] = y; key[hi] = x; }
            }
            __syncthreads();
        }
    }

    int n_take = 0;
    if (a.mode == SPOT_MODE_TOPK) {
        n_take = min(max(0, a.top_k - n_reserved), n_res);
        if (a.probs) {
            for (int j = tid; j < n_b; j += SEL_THREADS) a.probs[(int64_t)row * a.nb_stride + j] = 0.f;
        }
    } else {
        // Eq. 7 in fp64 on the sorted residual blocks; z = s_bar / T; m = z of rank 0.
        const int per = (n + SEL_THREADS - 1) / SEL_THREADS;      // consecutive ranks per thread (<= 8)
        const int r0 = tid * per;
        double zmax = 0.0;
        if (n_res > 0) zmax = (double)from_orderable(~(uint32_t)(key[0] >> 32)) / a.temperature;
        double e[8];
        double loc = 0.0;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            e[u] = 0.0;
            int r = r0 + u;
            if (u < per && r < n_res) {
                double z = (double)from_orderable(~(uint32_t)(key[r] >> 32)) / a.temperature;
                e[u] = exp(z - zmax);
            }
            loc += e[u];
        }
        double total;
        block_inclusive_scan(loc, wtot, &total);
        __syncthreads();
        // p~ = e / sum, then the prefix mass along the sorted order
        double pl = 0.0;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            e[u] = (total > 0.0) ? e[u] / total : 0.0;
            pl += e[u];
        }
        double dummy;
        double incl = block_inclusive_scan(pl, wtot, &dummy);
        double run = incl - pl;
        int below = 0;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            int r = r0 + u;
            if (u < per && r < n_res) {
                run += e[u];
                mass[r] = e[u];
                if (run < a.p) ++below;              // ranks whose cumulative mass is still < p
            }
        }
        if (below) atomicAdd(&s_nstar, below);
        __syncthreads();
        int n_star;
        if (n_res == 0) n_star = 0;
        else if (a.p >= 1.0) n_star = n_res;
        else n_star = min(n_res, s_nstar + 1);
        n_take = n_star;
        int target = min(a.kmin, n_b);
        if (n_reserved + n_take < target) n_take = min(n_res, target - n_reserved);
        if (a.probs) {
            float* pr = a.probs + (int64_t)row * a.nb_stride;
            for (int j = tid; j < n_b; j += SEL_THREADS)
                if (!(j >= sink_end && j < rec_beg)) pr[j] = 0.f;
            for (int r = tid; r < n_res; r += SEL_THREADS) pr[(uint32_t)key[r]] = (float)mass[r];
        }
    }
    for (int r = tid; r < n_take; r += SEL_THREADS) flag[(uint32_t)key[r]] = 1;
    __syncthreads();

    // ascending compaction of the selected block ids
    const int per = (n + SEL_THREADS - 1) / SEL_THREADS;
    const int j0 = tid * per;
    int cnt = 0;
    for (int u = 0; u < per; ++u) {
        int j = j0 + u;
        if (j < n_b && flag[j]) ++cnt;
    }
    int total_sel;
    int incl = block_inclusive_scan_int(cnt, itot, &total_sel);
    int pos = incl - cnt;
    int32_t* out = a.indices + (int64_t)row * a.cap;
    for (int u = 0; u < per; ++u) {
        int j = j0 + u;
        if (j < n_b && flag[j]) {
            if (pos < a.cap) out[pos] = j;
            ++pos;
        }
    }
    for (int j = total_sel + tid; j < a.cap; j += SEL_THREADS) out[j] = -1;
    if (tid == 0) a.budgets[row] = min(total_sel, a.cap);
}

}  // namespace

spot_status run_select(const spot_select_params* p, const float* scores, int nb_stride, int rows_per_seq,
                       int max_nb, cudaStream_t s) {
    if (max_nb > SEL_MAX_NB) return SPOT_ERR_UNSUPPORTED;
    int n = 1;
    while (n < max_nb) n <<= 1;
    SelectArgs a;
    a.scores = scores; a.nb_stride = nb_stride; a.seq_len = p->seq_len; a.n_q = rows_per_seq;
    a.q_start = p->q_start; a.q_block = p->q_block; a.blk = p->blk;
    a.mode = p->mode; a.top_k = p->top_k; a.p = p->p; a.temperature = p->temperature;
    a.sink = p->sink_blocks; a.rec = p->recency_blocks; a.kmin = p->kmin_blocks;
    a.indices = p->indices; a.cap = p->cap; a.budgets = p->budgets; a.probs = p->block_probs;
    size_t smem = (size_t)n * 17;
    static bool attr_set = false;
    if (!attr_set) {
        SPOT_CUDA_TRY(cudaFuncSetAttribute(select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SEL_MAX_NB * 17));
        attr_set = true;
    }
    select_kernel<<<(unsigned)(p->B * rows_per_seq), SEL_THREADS, smem, s>>>(a, n);
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}

}  // namespace spot
