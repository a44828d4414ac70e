// Step a2, histogram partition (rows of up to 2048 blocks; up to 8192 with 1024 threads x 8 keys) -- reserved tier, residual softmax (Eq. 7), nucleus +
// K_min floor (Eq. 8) or static top-K (Eq. 6), one CTA of 1024 threads x 2 keys (decode) or 256 threads x 8 keys (prefill) per selection row.
//
// The rule only needs (a) the mass in front of the cut and (b) the key value tau at the cut, not a full sort.  So:
//   1. keys (order-preserving 32-bit images of the scores, ascending key = descending score) go into as many bins as the row has slots by a
//      MONOTONE map of the key range (float multiply + truncate), i.e. bins are contiguous key ranges in rank order;
//   2. an exclusive scan of the bin counts turns the bins into rank ranges, and a counting-sort scatter groups
//      (key, exp(z - z_max)) by bin in shared memory -- unordered inside a bin, exactly ordered across bins;
//   3. a prefix sum of the masses in that grouped order is exact at every bin boundary, so the first position whose
//      running mass reaches p * total names the bin that holds the cut;
//   4. only that bin (typically 1-3 blocks) is ranked exactly -- by one warp when it holds <= 32 keys, by a plain
//      counting pass of the whole CTA otherwise (degenerate inputs such as all-equal scores take an arithmetic
//      shortcut) -- which gives n* and tau; K_min / top-K ask the same machinery for "the key of rank r";
//   5. blocks with a better key than tau are selected, blocks tied with tau are taken in ascending block index until
//      the count is reached (R7), and the ascending index list falls out of a ballot/popc scan in index order.
// exp, normalisation and the running mass are fp64 (the fp32 block score is then the only source of disagreement
// with the fp64 oracle).  ~12 CTA barriers and 2300 instructions per warp instead of a 66-step
// bitonic network and 3400.  With 256 threads x 8 keys the launch was 13.9 us against 14.1 us at n_b = 2048 all the same:
// a kernel that runs once per step on 4 SMs from cold caches is a chain of latencies (instruction fetch, two dependent
// DRAM misses, eight sequential fp64 exps per thread), not of work.  1024 threads x 2 keys shorten every per-thread
// section: decode step 172.6 -> 169 us (profiles/r1_decode_cfg3_launches.md, D).
#include "select_common.cuh"

namespace spot {

namespace {

// SH_N keys per row (2048, or 8192 for the long rows of 16-token blocks / L > 128K) and as many bins
template <int SH_NBIN>
struct BinMap {
    uint32_t kmn;
    float scale;
    __device__ __forceinline__ int operator()(uint32_t key) const {
        const int b = (int)((float)(key - kmn) * scale);      // monotone in key
        return b < SH_NBIN - 1 ? b : SH_NBIN - 1;
    }
};

// Exact ranking of one bin by a single warp (cB <= 32 keys at grouped positions sB ..).  by_mass: returns the number
// n_in of keys (in rank order) whose running mass base + ... is still < target, clamped to cB - 1; else n_in = want.
// tau = key of rank n_in inside the bin.  Equal keys are ranked by position (they carry equal mass).
__device__ __forceinline__ void warp_resolve(const uint32_t* s_k, const double* s_e, int sB, int cB, double base,
                                             double target, int want, bool by_mass, int lane, int& n_in, uint32_t& tau) {
    const uint32_t k = lane < cB ? s_k[sB + lane] : KEY_PAD;
    const double e = (by_mass && lane < cB) ? s_e[sB + lane] : 0.0;
    int rank = 0;
    for (int j = 0; j < cB; ++j) {
        const uint32_t kj = __shfl_sync(0xffffffffu, k, j);
        rank += (kj < k || (kj == k && j < lane)) ? 1 : 0;
    }
    if (lane >= cB) rank = 64 + lane;
    n_in = want;
    if (by_mass) {
        double acc = base, mine = 0.0;
        for (int r = 0; r < cB; ++r) {
            const int src = __ffs(__ballot_sync(0xffffffffu, rank == r)) - 1;
            acc += __shfl_sync(0xffffffffu, e, src);
            if (rank == r) mine = acc;
        }
        n_in = __popc(__ballot_sync(0xffffffffu, lane < cB && mine < target));
    }
    n_in = max(0, min(n_in, cB - 1));
    const int src = __ffs(__ballot_sync(0xffffffffu, rank == n_in)) - 1;
    tau = __shfl_sync(0xffffffffu, k, src);
}

// E keys per thread, SH_N / E threads: decode rows (a handful of CTAs, pure latency) run 1024 threads x 2 keys so that
// every per-thread section (two fp64 exps instead of eight, ...) is short; prefill rows (a thousand CTAs, throughput) run
// 256 threads x 8 keys.
// (rows of up to 2048 keys keep their 32 KiB of arrays static; the 8192-key form takes 128 KiB of dynamic shared memory)
template <int SH_N, int SH_E>
__global__ void __launch_bounds__(SH_N / SH_E) select_hist_kernel(SelectArgs a) {
    constexpr int SH_T = SH_N / SH_E, SH_WARPS = SH_T / 32, SH_NBIN = SH_N;
    constexpr bool STATIC = SH_N <= 2048;
    constexpr int PK_SHIFT = SH_N > 4096 ? 13 : 12;           // bin << PK_SHIFT | rank inside the bin
    __shared__ uint32_t st_cnt[STATIC ? SH_NBIN : 1];
    __shared__ double st_e[STATIC ? SH_N : 1];
    __shared__ uint32_t st_k[STATIC ? SH_N : 1];
    extern __shared__ __align__(16) unsigned char sh_dyn[];
    double* const s_e = STATIC ? st_e : reinterpret_cast<double*>(sh_dyn);                           // masses grouped by bin
    uint32_t* const s_k = STATIC ? st_k : reinterpret_cast<uint32_t*>(sh_dyn + SH_N * 8);            // keys grouped by bin
    uint32_t* const s_cnt = STATIC ? st_cnt : reinterpret_cast<uint32_t*>(sh_dyn + SH_N * 12);       // bin counts, then exclusive starts
    __shared__ double s_wd[SH_WARPS];
    __shared__ uint32_t s_wu[SH_WARPS][2];
    __shared__ int s_wi[SH_WARPS][2];
    __shared__ int s_seg[SH_N / 32][2];
    __shared__ double s_base;
    __shared__ uint32_t s_tau;
    __shared__ int s_nin, s_tot[2];

    const int row = blockIdx.x;
    const int b = row / a.n_q, i = row - b * a.n_q;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool piped = a.sync.tag != 0u;
    SPOT_STAMP(a.sync, 1, 0);
    if (piped) pdl_launch_dependents();
    // A pipelined call runs the body twice: first DRY, on a synthetic row with every global store off, while the row's
    // block scores are still being produced -- this kernel's 45 KB of code (and the constants of the fp64 exp) come from
    // DRAM, behind an HBM stream at full rate (the bench flushes L2 before every step), and a cold pass costs 10-13 us
    // there against 8-10 us from warm caches.  The selection CTA has its SM to itself and nothing else to do -- but only
    // rows whose scores are still far off (dry_from_row, estimated on the host from the bytes in front of them) take it:
    // a row that is ready before the dry pass ends would only wait for it.
#pragma unroll 1
  for (int pass = (piped && b >= a.dry_from_row) ? 0 : 1; pass < 2; ++pass) {
    const bool dry = pass == 0;
    float sraw[SH_E];
    int n_b;
    if (dry) {
        n_b = min(SH_N, a.tagged_stride);
#pragma unroll
        for (int r = 0; r < SH_E; ++r) {
            const uint32_t j = (uint32_t)(warp * (32 * SH_E) + lane + 32 * r);
            sraw[r] = (float)((j * 2654435761u) >> 8) * (8.0f / 16777216.0f);      // scores spread over [0, 8)
        }
    } else if (piped) {
        // pipelined step (decode rows): this CTA is resident BESIDE the scoring kernel and waits for its own sequence only
        // -- every block score arrives as one {tag, fp32 bits} word; an entry is re-read until it carries this call's tag,
        // then cleared (common.cuh, StepSync)
        n_b = min((min(max(a.seq_len[b], 0), a.max_len) + a.blk - 1) / a.blk, SH_N);
        unsigned long long* trow = a.tagged + (int64_t)row * a.tagged_stride;
        unsigned long long v[SH_E];
#pragma unroll
        for (int r = 0; r < SH_E; ++r) {
            const int j = warp * (32 * SH_E) + lane + 32 * r;
            v[r] = j < n_b ? ld_tagged_score(trow + j) : ((unsigned long long)a.sync.tag << 32);
        }
#pragma unroll
        for (int r = 0; r < SH_E; ++r) {
            const int j = warp * (32 * SH_E) + lane + 32 * r;
            while ((uint32_t)(v[r] >> 32) != a.sync.tag) { __nanosleep(256); v[r] = ld_tagged_score(trow + j); }
            sraw[r] = __uint_as_float((uint32_t)v[r]);
            if (j < n_b) {
                trow[j] = (unsigned long long)(uint32_t)v[r];           // tag cleared: consumed
                if (a.scores_out) a.scores_out[(int64_t)row * a.nb_stride + j] = sraw[r];
            }
        }
        SPOT_STAMP(a.sync, 1, 1);
    } else {
        pdl_wait();
        pdl_launch_dependents();
        // the row's scores are requested before seq_len is known (two independent DRAM misses instead of a chain)
        const float* srow = a.scores + (int64_t)row * a.nb_stride;
#pragma unroll
        for (int r = 0; r < SH_E; ++r) {
            const int j = warp * (32 * SH_E) + lane + 32 * r;
            sraw[r] = j < a.nb_stride ? srow[j] : 0.f;
        }
        if (a.q_block == 1) n_b = (min(max(a.seq_len[b], 0), a.max_len) + a.blk - 1) / a.blk;
        else n_b = (a.q_start + (i + 1) * a.q_block - 1) / a.blk + 1;
    }
    n_b = min(n_b, SH_N);
    const int sink_end = min(a.sink, n_b);
    const int rec_beg = max(sink_end, n_b - a.rec);     // residual blocks: [sink_end, rec_beg)
    const int n_res = rec_beg - sink_end;
    const int n_reserved = n_b - n_res;
    const int ebase = warp * (32 * SH_E) + lane;                // block of register r: ebase + 32 r
    const bool topp = a.mode != SPOT_MODE_TOPK;

    // ---- load: block scores -> keys; key range of the residual blocks
    uint32_t okey[SH_E];
    uint32_t kmn = 0xffffffffu, kmx = 0u;
#pragma unroll
    for (int r = 0; r < SH_E; ++r) {
        const int j = ebase + 32 * r;
        const bool resid = j >= sink_end && j < rec_beg;
        okey[r] = resid ? score_key(sraw[r]) : KEY_PAD;
        if (resid) { kmn = min(kmn, okey[r]); kmx = max(kmx, okey[r]); }
        s_cnt[tid * SH_E + r] = 0u;
    }
    kmn = __reduce_min_sync(0xffffffffu, kmn);
    kmx = __reduce_max_sync(0xffffffffu, kmx);
    if (lane == 0) { s_wu[warp][0] = kmn; s_wu[warp][1] = kmx; }
    if (tid == 0) { s_nin = 0; s_tau = 0u; s_base = 0.0; }
    __syncthreads();
    SPOT_STAMP(a.sync, 4, 0);
    // (cross-warp combines: lane w reads warp w's word and the warp reduces -- a loop over the 32 warps in every thread
    // was 40 % of this kernel's instructions, and with 32 warps per SM the kernel is issue-bound)
    kmn = __reduce_min_sync(0xffffffffu, lane < SH_WARPS ? s_wu[lane][0] : 0xffffffffu);
    kmx = __reduce_max_sync(0xffffffffu, lane < SH_WARPS ? s_wu[lane][1] : 0u);

    int n_take = 0;
    uint32_t tau = 0u;
    double e[SH_E], total = 0.0;
#pragma unroll
    for (int r = 0; r < SH_E; ++r) e[r] = 0.0;

    if (n_res > 0) {
        BinMap<SH_NBIN> bin_of;
        bin_of.kmn = kmn;
        bin_of.scale = (float)SH_NBIN / ((float)(kmx - kmn) + 1.0f);
        // ---- masses (Eq. 7 numerators, fp64), bins, rank inside the bin
        // (x / 1.0 == x exactly: the default temperature, skips three fp64 divisions per thread)
        const bool t_one = a.temperature == 1.0;
        const double zmax = t_one ? (double)key_score(kmn) : (double)key_score(kmn) / a.temperature;
        // (one rolled loop -- the fp64 exp is ~150 instructions and this kernel runs once per step from a cold
        // instruction cache: code size, not instruction count, is what its latency is made of.  The arrays stay in
        // registers: every trip works on element 0 and rotates.)
        uint32_t pk[SH_E];                                   // bin << PK_SHIFT | rank inside the bin; 0xffffffff: not residual
        {
            uint32_t kq[SH_E];
#pragma unroll
            for (int r = 0; r < SH_E; ++r) { kq[r] = okey[r]; pk[r] = 0xffffffffu; }
#pragma unroll 1
            for (int r = 0; r < SH_E; ++r) {
                const int j = ebase + 32 * r;
                double ev = 0.0;
                uint32_t pv = 0xffffffffu;
                if (j >= sink_end && j < rec_beg) {
                    if (topp) {
                        const double x = (double)key_score(kq[0]);
                        ev = exp((t_one ? x : x / a.temperature) - zmax);
                    }
                    const int bn = bin_of(kq[0]);
                    pv = ((uint32_t)bn << PK_SHIFT) | atomicAdd(&s_cnt[bn], 1u);
                }
#pragma unroll
                for (int u = 0; u < SH_E - 1; ++u) { kq[u] = kq[u + 1]; e[u] = e[u + 1]; pk[u] = pk[u + 1]; }
                e[SH_E - 1] = ev;
                pk[SH_E - 1] = pv;
            }
        }
        __syncthreads();
        SPOT_STAMP(a.sync, 4, 1);
        // ---- exclusive scan of the bin counts: thread t owns bins 8t .. 8t+7
        {
            uint32_t c[SH_E], run = 0;
#pragma unroll
            for (int u = 0; u < SH_E; ++u) { c[u] = s_cnt[tid * SH_E + u]; run += c[u]; }
            uint32_t inc = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane == 31) s_wi[warp][0] = (int)inc;
            __syncthreads();
            uint32_t off = inc - run;
            off += __reduce_add_sync(0xffffffffu, (lane < SH_WARPS && lane < warp) ? (uint32_t)s_wi[lane][0] : 0u);
#pragma unroll
            for (int u = 0; u < SH_E; ++u) { s_cnt[tid * SH_E + u] = off; off += c[u]; }
        }
        __syncthreads();
        // ---- counting-sort scatter: grouped by bin, bins in rank order
#pragma unroll
        for (int r = 0; r < SH_E; ++r)
            if (pk[r] != 0xffffffffu) {
                const int pos = (int)s_cnt[pk[r] >> PK_SHIFT] + (int)(pk[r] & ((1u << PK_SHIFT) - 1u));
                s_k[pos] = okey[r];
                if (topp) s_e[pos] = e[r];
            }
        __syncthreads();
        SPOT_STAMP(a.sync, 4, 2);
        // ---- what has to be resolved exactly: up to two queries against one bin each, run by ONE copy of the code
        //      query 0 (dual top-p, p < 1): the bin holding the cut of the running mass -> n*, tau
        //      query 1 (top-K, K_min floor): the key of rank n_take - 1
        double target = 0.0, off = 0.0, c[SH_E];
        int n_lt = 0;
        if (topp) {
            // running mass in grouped order: thread t owns positions 8t .. 8t+7
            double run = 0.0;
#pragma unroll
            for (int u = 0; u < SH_E; ++u) {
                const int pos = tid * SH_E + u;
                run += pos < n_res ? s_e[pos] : 0.0;
                c[u] = run;
            }
            double inc = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const double t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane == 31) s_wd[warp] = inc;
            __syncthreads();
            off = inc - run;
            {
                const double wv = lane < SH_WARPS ? s_wd[lane] : 0.0;
                double before = lane < warp ? wv : 0.0, all = wv;
#pragma unroll
                for (int o = 16; o; o >>= 1) {
                    before += __shfl_xor_sync(0xffffffffu, before, o);
                    all += __shfl_xor_sync(0xffffffffu, all, o);
                }
                off += before;
                total = all;
            }
            target = a.p * total;
            int cnt = 0;
#pragma unroll
            for (int u = 0; u < SH_E; ++u) cnt += (tid * SH_E + u < n_res && off + c[u] < target) ? 1 : 0;
            cnt = __reduce_add_sync(0xffffffffu, cnt);
            if (lane == 0) s_wi[warp][1] = cnt;
            __syncthreads();
            n_lt = __reduce_add_sync(0xffffffffu, lane < SH_WARPS ? s_wi[lane][1] : 0);
            n_take = n_res;                                   // p >= 1: all of B_res by definition (R20)
        } else {
#pragma unroll
            for (int u = 0; u < SH_E; ++u) c[u] = 0.0;
            n_take = min(max(0, a.top_k - n_reserved), n_res);
        }
        bool have_tau = false;
#pragma unroll 1
        for (int query = (topp && a.p < 1.0) ? 0 : 1; query < 2; ++query) {
            const bool by_mass = query == 0;
            if (!by_mass) {
                if (have_tau || n_take <= 0) break;
                if (n_take == n_res) { tau = kmx; break; }    // everything: the worst key
            }
            const int B = bin_of(s_k[by_mass ? min(n_lt, n_res - 1) : n_take - 1]);   // the bin holding that position
            const int sB = (int)s_cnt[B];
            const int cB = (B + 1 < SH_NBIN ? (int)s_cnt[B + 1] : n_res) - sB;
            const int want = n_take - 1 - sB;
            if (by_mass && sB > 0 && tid == ((sB - 1) / SH_E)) {   // running mass in front of the bin: its owner publishes it
                double v = c[0];
#pragma unroll
                for (int u = 1; u < SH_E; ++u) v = (((sB - 1) % SH_E) == u) ? c[u] : v;
                s_base = off + v;
            }
            __syncthreads();
            const double base = (by_mass && sB > 0) ? s_base : 0.0;
            // exact ranking of the bin (grouped positions sB .. sB + cB - 1): s_nin = keys of the bin in front of the
            // cut (or `want`), s_tau = the key of that rank
            if (cB <= 32) {
                if (warp == 0) {
                    int n_in;
                    uint32_t t;
                    warp_resolve(s_k, s_e, sB, cB, base, target, want, by_mass, lane, n_in, t);
                    if (lane == 0) { s_nin = n_in; s_tau = t; }
                }
            } else {
                // a crowded bin (degenerate score distributions): whole CTA
                uint32_t lo = 0xffffffffu, hi = 0u;
                for (int x = tid; x < cB; x += SH_T) { const uint32_t k = s_k[sB + x]; lo = min(lo, k); hi = max(hi, k); }
                lo = __reduce_min_sync(0xffffffffu, lo);
                hi = __reduce_max_sync(0xffffffffu, hi);
                if (lane == 0) { s_wu[warp][0] = lo; s_wu[warp][1] = hi; }
                if (tid == 0) s_nin = 0;
                __syncthreads();
                lo = __reduce_min_sync(0xffffffffu, lane < SH_WARPS ? s_wu[lane][0] : 0xffffffffu);
                hi = __reduce_max_sync(0xffffffffu, lane < SH_WARPS ? s_wu[lane][1] : 0u);
                if (lo == hi) {
                    // every key of the bin is the same: equal masses, ranked by position -> arithmetic
                    if (tid == 0) {
                        int m = want;
                        if (by_mass) {
                            const double e0 = s_e[sB];
                            m = e0 > 0.0 ? (int)fmin(fmax(ceil((target - base) / e0) - 1.0, 0.0), (double)(cB - 1)) : 0;
                            while (m > 0 && base + (double)m * e0 >= target) --m;
                            while (m < cB - 1 && base + (double)(m + 1) * e0 < target) ++m;
                        }
                        s_nin = max(0, min(m, cB - 1));
                        s_tau = lo;
                    }
                } else {
                    // Sort the bin's (key, mass) pairs by key, in place: a bitonic network in its all-ascending form (first
                    // sub-step of every block size compares i with i ^ (k - 1), the others i with i ^ j), so that positions
                    // past cB act as +inf padding and a comparator that reaches one is a no-op.  Equal keys carry equal masses
                    // and ties are broken by BLOCK INDEX at emission, from the threshold key alone -- the order of equal keys
                    // inside the bin decides nothing, and nothing after this reads the bin in its scattered order.  Then the
                    // cut is a prefix sum over the sorted masses and the threshold the key at that rank.  (Until the end of
                    // round 2 this was two O(cB^2 / threads) counting passes: one block of score exactly 0 beside 8191 scores
                    // within 1e-3 of each other put every residual key into one bin and the row took 5.9 ms.)
                    for (int k = 2; (k >> 1) < cB; k <<= 1) {
                        bool first = true;
                        for (int jj = k >> 1; jj > 0; jj >>= 1, first = false) {
                            const int mask = first ? k - 1 : jj;
                            for (int x = tid; x < cB; x += SH_T) {
                                const int y = x ^ mask;
                                if (y > x && y < cB) {
                                    const uint32_t kx = s_k[sB + x], ky = s_k[sB + y];
                                    if (kx > ky) {
                                        s_k[sB + x] = ky; s_k[sB + y] = kx;
                                        const double ex = s_e[sB + x];
                                        s_e[sB + x] = s_e[sB + y]; s_e[sB + y] = ex;
                                    }
                                }
                            }
                            __syncthreads();
                        }
                    }
                    int n_in = want;
                    if (by_mass) {
                        // keys in front of the cut: running mass (inclusive, fp64) still below the target
                        const int per = (cB + SH_T - 1) / SH_T;
                        const int x0 = min(tid * per, cB), x1 = min(x0 + per, cB);
                        double loc = 0.0;
                        for (int x = x0; x < x1; ++x) loc += s_e[sB + x];
                        double inc = loc;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const double up = __shfl_up_sync(0xffffffffu, inc, o);
                            if (lane >= o) inc += up;
                        }
                        if (lane == 31) s_wd[warp] = inc;
                        __syncthreads();
                        double cum = base;
                        for (int w = 0; w < warp; ++w) cum += s_wd[w];
                        cum += inc - loc;
                        int cnt = 0;
                        for (int x = x0; x < x1; ++x) { cum += s_e[sB + x]; cnt += cum < target ? 1 : 0; }
                        cnt = __reduce_add_sync(0xffffffffu, cnt);
                        if (lane == 0 && cnt) atomicAdd(&s_nin, cnt);
                        __syncthreads();
                        n_in = s_nin;
                        __syncthreads();
                    }
                    n_in = max(0, min(n_in, cB - 1));
                    if (tid == 0) { s_tau = s_k[sB + n_in]; s_nin = n_in; }
                }
            }
            __syncthreads();
            tau = s_tau;
            have_tau = true;
            if (by_mass) {
                n_take = sB + s_nin + 1;                      // n*
                const int floor_cnt = min(a.kmin, n_b);       // K_min floor on the union (R8)
                if (n_reserved + n_take < floor_cnt) { n_take = min(n_res, floor_cnt - n_reserved); have_tau = false; }
            }
            __syncthreads();                                  // s_nin / s_tau may be rewritten by the next query
        }
    }
    __syncthreads();
    SPOT_STAMP(a.sync, 4, 3);

    // ---- index order: A = reserved or strictly better than tau (certainly selected), Tt = tied with tau
    constexpr int NSEG = SH_N / 32;                       // 32-block segments: (warp, register)
    int prefA[SH_E], prefT[SH_E];
    uint32_t isA = 0, isT = 0;
#pragma unroll
    for (int r = 0; r < SH_E; ++r) {
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
        if (lane == 0) { s_seg[warp * SH_E + r][0] = __popc(ba); s_seg[warp * SH_E + r][1] = __popc(bt); }
    }
    __syncthreads();
    if (warp == 0) {
        constexpr int PER = NSEG / 32;
        int va[PER], vt[PER], ra = 0, rt = 0;
#pragma unroll
        for (int u = 0; u < PER; ++u) {
            const int s = lane * PER + u;
            va[u] = s_seg[s][0];
            vt[u] = s_seg[s][1];
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
            s_seg[s][0] = oa; s_seg[s][1] = ot;
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
    for (int r = 0; r < SH_E; ++r) {
        const int j = ebase + 32 * r;
        const int a_before = s_seg[warp * SH_E + r][0] + prefA[r];
        const int t_before = s_seg[warp * SH_E + r][1] + prefT[r];
        int pos = -1;
        if ((isA >> r) & 1u) pos = a_before + min(t_before, need);
        else if (((isT >> r) & 1u) && t_before < need) pos = a_before + t_before;
        if (pos >= 0 && pos < a.cap && !dry) out[pos] = j;
    }
    if (!dry) {
        for (int j = total_sel + tid; j < a.cap; j += SH_T) out[j] = -1;
        if (tid == 0) a.budgets[row] = min(total_sel, a.cap);
    }

    if (a.probs && !dry) {
        float* pr = a.probs + (int64_t)row * a.nb_stride;
        const double inv_total = total > 0.0 ? 1.0 / total : 0.0;
#pragma unroll
        for (int r = 0; r < SH_E; ++r) {
            const int j = ebase + 32 * r;
            if (j < n_b) pr[j] = (float)(e[r] * inv_total);      // 0 on reserved blocks and in top-K mode
        }
    }
    __syncthreads();                                  // (the shared arrays are reused by the next pass)
  }
    if (piped) {
        __syncthreads();                              // the row's list, budget and probabilities are written
        SPOT_STAMP(a.sync, 1, 2);
        if (tid == 0) {
            if (a.sync.ready) { __threadfence(); st_release_u32(a.sync.ready + b, a.sync.tag); }
            // completion of this grid implies completion of the scoring grid -- through its LAST CTA alone: the others
            // must leave their SM to the selection CTAs queued behind them (B > SMs left to this kernel)
            if (blockIdx.x == gridDim.x - 1) pdl_wait();
        }
    }
}

}  // namespace

spot_status launch_select_hist(const SelectArgs& a, int rows, int max_nb, cudaStream_t s) {
    if (max_nb > 2048) {
        constexpr int BIG = 8192, BIG_SMEM = BIG * 16;
        static unsigned long long smem_attr_done = 0;
        SPOT_CUDA_TRY(set_max_smem_once(select_hist_kernel<BIG, 8>, BIG_SMEM, smem_attr_done));
        SPOT_CUDA_TRY(launch_pdl(select_hist_kernel<BIG, 8>, dim3((unsigned)rows), dim3(BIG / 8), BIG_SMEM, s, a));
    } else if (rows <= 32) {
        SPOT_CUDA_TRY(launch_pdl(select_hist_kernel<2048, 2>, dim3((unsigned)rows), dim3(2048 / 2), 0, s, a));
    } else {
        SPOT_CUDA_TRY(launch_pdl(select_hist_kernel<2048, 8>, dim3((unsigned)rows), dim3(2048 / 8), 0, s, a));
    }
    return SPOT_OK;
}

}  // namespace spot
