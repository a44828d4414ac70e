// Step a1', prefill form -- one score per (64-query block, 64-key block) tile (reading R2):
//   s_bar[i,j] = max_{q in i} max_{t in j, t <= q}  sum_h w_h[q] ReLU(q^I_h[q] . k^I_{h,t}).
//
// This IS a dense contraction (4 heads x [Tq x 64] x [64 x L_visible]), so it runs on the 5th-gen tensor cores:
//   * one persistent CTA per SM; the unit of work is a STEP = (128-query tile = two query blocks, PAIR of key blocks), and
//     every CTA gets a contiguous range of the same number of steps (ItemWalk below);
//   * warp 8 lane 0: TMA producer -- the query tile ([4 heads][128][64] BF16, 64 KiB) and a 2-stage ring of key-block
//     PAIRS ([4 heads][128 keys][64], 64 KiB) land in 128-byte-swizzled shared memory through 4-D tensor maps;
//   * warp 9 (converged, one elected lane issues): tcgen05.mma with M = 128 queries, N = 128 keys (two key blocks), K = 16: four k-steps per
//     head into a 128-column TMEM accumulator.  N = 64 made every MMA read 6 KiB of operands for 16 cycles of math
//     (384 B/clk) and the tensor pipe sat at 65 % busy for 37 % of peak (profiles/r1_prefill_cfg5.md); N = 128 halves
//     the A-operand re-reads per flop.  The 512 TMEM columns are a ring of FOUR accumulators, one per (pair, head):
//     the issuer runs up to three heads ahead of the epilogue;
//   * warps 0-7: epilogue.  Warp w owns TMEM lanes 32 (w & 3) .. +31 (one query per lane) and the 64 columns of key
//     block (w >> 2) of the pair.  Head by head it reads the accumulator (two 32-column tcgen05.ld, the next one in
//     flight under the arithmetic on the previous), releases it, and adds w_h ReLU(d_h) to a 64-register running sum; after the fourth head the tile maximum is a REDUX.MAX over an
//     order-preserving integer key plus one shared-memory atomicMax per warp.
// The epilogue is the near-co-bound (9 lane-ops per (query, key) pair against 512 tensor flops), so ReLU is split
// between the two fp32 pipes: heads 0-1 use (w/2)(d + |d|) (FADD with an abs modifier, FMA pipe), heads 2-3 use
// w max(d, 0) (ALU pipe); both forms give bit-identical products.  The weighted sum uses packed FFMA2, head 0's product
// packed FMUL2 (cfg5 GEMM alone: BF16 1.086 -> 1.03 ms, FP8 1.004 -> 0.986, MXFP4 1.031 -> 1.014).
#include "common.cuh"
#include "tc100.cuh"

#include <string.h>

namespace spot {

#ifdef SPOT_TRACE
long long* g_pf_trace = nullptr;      // development builds only
#endif

namespace {

constexpr int PF_H = 4;                 // selector heads
constexpr int PF_M = 128;               // queries per tile (two 64-query blocks)
constexpr int PF_N = 128;               // keys per MMA (two 64-key blocks)
constexpr int PF_CHUNK = 32;            // key blocks per work item
constexpr int PF_EPI_WARPS = 8;
constexpr uint32_t PF_PLANE_BYTES = 128 * 64 * 2;          // [128 rows][64 d] BF16: one 128-byte swizzle row per token
constexpr uint32_t PF_SMEM_MISC = 2048;        // barriers, TMEM slot, tile maxima [CHUNK][4 quarters][2 query blocks]

// Geometry in BYTES per head row (HB), because that is all the tensor pipe and the TMA see: a token's selector row is
// PF_H heads x HB bytes, cut into 128-byte planes (one 128-byte swizzle row per token per plane).
//   HB = 128 : BF16 d_idx = 64, or FP8-E4M3 d_idx = 128 -- a head is one plane; a K slot holds all four heads of a
//              key-block pair (64 KiB, 2 slots beside the 64 KiB query tile); four 32-byte k-steps per head.
//   HB = 256 : BF16 d_idx = 128 (the paper's selector width) -- a head is two planes; a K slot holds ONE head
//              of a pair (32 KiB, 3 slots beside the 128 KiB query tile) and the issuer accumulates 8 k-steps.
//   HB = 64  : FP8-E4M3 d_idx = 64 -- two heads share a plane (32 KiB query tile, six 32 KiB slots); a head is the two k-steps at byte
//              (h & 1) * 64 of its plane.
// F8 (f2, round 2): both operands are FP8-E4M3 bytes straight from the cache layout (`tcgen05.mma kind::f8f6f4`, K = 32
// elements = 32 bytes per instruction, fp32 accumulate in TMEM); the BF16 forms use kind::f16 (K = 16 elements = 32 bytes).
// The TMA map describes bytes as BF16 pairs either way.
//
// Round-2 measurements that shaped this (per-CTA clock64 timeline of producer / issuer / epilogue, _work-side probes; DESIGN.md
// section 7): (1) under `if (lane == 0)` ptxas wraps every tcgen05.mma in an ELECT / BRA.U.ANY loop of its own, one basic
// block per MMA, and the issuing thread needed 70-130 cycles per 64-cycle MMA -- the issuer warp now runs converged and one
// ELECTED lane issues (tc100.cuh, umma_*_elect): 140-190 cycles per head of four MMAs; (2) the epilogue keeps one 32-column
// tcgen05.ld in flight under the arithmetic on the previous one; (3) the query tile as the A operand in TENSOR MEMORY
// (tcgen05.mma with [a_tmem]) halves the shared-memory reads of the MMAs and frees 64-128 KiB for a deeper key ring, but
// costs accumulators (3 instead of 4 at HB = 128, 2 at HB = 256) and was 19 % / 8 % SLOWER: the depth of the accumulator ring
// is what hides the issuer <-> epilogue hand-off, so both operands stay in shared memory; (4) a thread-block cluster of two
// query tiles sharing every key load by TMA multicast, a key ring of ten 16 KiB single-head slots, sixteen epilogue warps,
// and both fp32 pipes inside every head (element 0 of a pair through FADD, element 1 through FMNMX) were all measured
// equal or slower.
// MX4 (f2, round 2): both operands are MXFP4 straight from the opaque cache layout (quantize.cu) -- a token row of packed
// E2M1 codes is PF_H * HB bytes with HB = 32 (d_idx 64) or 64 (d_idx 128), one 128-byte swizzle row per 128 bytes, and
// `tcgen05.mma kind::mxf4.block_scale.block32` multiplies in the UE8M0 group scales itself (K = 64 elements = 32 bytes per
// instruction, two scales per row and instruction).  The scales travel beside the codes (plain bulk copies of the tiles'
// scale rows into the tail of the slot) and four extra warps (one per TMEM lane quarter) move them into tensor memory in
// the layout the MMA reads (tc100.cuh) -- 16 columns for the query tile, 16 per key slot, which leaves room for a ring of
// THREE accumulators.
constexpr int PF_BF16 = 0, PF_F8 = 1, PF_MX4 = 2;
template <int HB, int KIND>
struct PfCfg {
    static constexpr bool F8 = KIND == PF_F8, MX4 = KIND == PF_MX4;
    static_assert(HB == 32 || HB == 64 || HB == 128 || HB == 256, "head row of 32, 64, 128 or 256 bytes");
    static_assert(MX4 ? (HB == 32 || HB == 64) : F8 ? (HB == 64 || HB == 128) : (HB == 128 || HB == 256),
                  "BF16: d_idx 64 / 128; FP8: d_idx 64 / 128; MXFP4: d_idx 64 / 128");
    static constexpr int PLANES = PF_H * HB / 128;                        // planes per token row
    static constexpr int KSTEPS = HB / 32;                                // 32-byte k-steps per head
    static constexpr bool PER_HEAD = HB == 256;                           // K ring granularity
    static constexpr int HEAD_PLANES = HB / 128;                          // planes per head (PER_HEAD only)
    static constexpr int STAGE_PLANES = PER_HEAD ? HEAD_PLANES : PLANES;  // planes of one K ring slot
    static constexpr int NG = MX4 ? PF_H * HB / 16 : 0;                   // MX4: scale bytes per token (8 / 16)
    static constexpr uint32_t SF_BYTES = MX4 ? 2048u : 0u;                // room for [128 rows][NG] scale bytes behind the codes
    static constexpr uint32_t Q_CODE_BYTES = PLANES * PF_PLANE_BYTES;
    static constexpr uint32_t K_CODE_BYTES = STAGE_PLANES * PF_PLANE_BYTES;
    static constexpr uint32_t Q_TILE_BYTES = Q_CODE_BYTES + SF_BYTES;
    static constexpr uint32_t K_STAGE_BYTES = K_CODE_BYTES + SF_BYTES;
    static constexpr int KSTAGES = MX4 ? 4 : (int)((224u * 1024u - Q_TILE_BYTES) / K_STAGE_BYTES);   // 2 / 3 / 6
    static_assert(KSTAGES >= 2 && KSTAGES <= 8, "key ring");
    static constexpr uint32_t SMEM_TILES = Q_TILE_BYTES + KSTAGES * K_STAGE_BYTES;
    static constexpr uint32_t SMEM_BYTES = 1024 + SMEM_TILES + PF_SMEM_MISC;   // 1024: manual alignment slack
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
    // (three accumulators instead of four cost the FP8 kernel 6 %: 1.065 against 1.004 ms at cfg5)
    static constexpr int NACC = MX4 ? 3 : 512 / PF_N;                     // TMEM: a ring of 128-column accumulators
    static constexpr int SF_WARPS = MX4 ? 4 : 0;
    // MX4: 16 warps = four warpgroups, so that the register file can be re-cut between the roles (setmaxnreg works on
    // whole warpgroups): 448 threads under one launch bound left the epilogue 128 registers and ~300 bytes of spills
    // (tile-score GEMM 1.46 ms against FP8's 1.00 ms); warps 14-15 only take part in the barriers
    static constexpr int THREADS = MX4 ? 512 : (PF_EPI_WARPS + 2) * 32;
    // MX4 tensor-memory columns behind the accumulators: the query tile's scale words, then one block per key slot
    static constexpr uint32_t SFQ_COL = NACC * PF_N, SFK_COL = SFQ_COL + 16;
    static_assert(!MX4 || SFK_COL + 16 * KSTAGES <= 512, "tensor memory");
    // shared-memory byte offset of k-step ks of head h inside a tile of planes [plane][128 rows][128 B]
    static constexpr uint32_t koff(int h, int ks) {
        return (uint32_t)((h * HB + ks * 32) / 128) * PF_PLANE_BYTES + (uint32_t)((h * HB + ks * 32) % 128);
    }
};

struct PrefillScoreArgs {
    const float* w;           // [B][Tq][4]
    float* scores;            // [B * n_qb][nb_stride]
    int nb_stride;
    int B, Tq, n_qb, n_qt;    // query blocks / query tiles per sequence
    int qb_start;             // q_start / 64
    int64_t total_steps;      // B * steps_per_seq (ItemWalk)
    int64_t steps_per_seq;
    int fine;                 // blk == 16 (f3): four scores per 64-key block, one per 16-token quarter
    // rows form (f4, the student's pass 1 of spot_train_kl; B = 1, q_start = 0): instead of one score per (query block, key
    // block) every QUERY gets, per 64-key block j it can see, the maxima of its blk-token blocks (row_blk[q][j * 64 / blk ..])
    // and the pair (max, sum exp(s - max)) over the block's visible keys (row_part[j][q]: a log-sum-exp in pieces)
    float* row_blk;           // nullptr: the tile-score form
    float2* row_part;         // [Tq / 64][Tq]
    int row_stride, row_blk_tokens;
    // MX4: the two caches (queries: a cache of Tq tokens per sequence) for the bulk copies of the scale rows
    const uint8_t* q_cache;
    const uint8_t* k_cache;
    int q_tiles, k_tiles;     // 64-token tiles per sequence
#ifdef SPOT_TRACE
    long long* trace;         // development builds only: [6 roles][2048 events] clock64 of CTA 5
#endif
};
#ifdef SPOT_TRACE
#define PF_STAMP(role, idx) do { if (a.trace && blockIdx.x == 5 && (idx) < 2048) a.trace[(role) * 2048 + (idx)] = clock64(); } while (0)
#else
#define PF_STAMP(role, idx) do { } while (0)
#endif

// contiguous global -> shared bulk copy (bytes a multiple of 16), completion counted on an mbarrier
__device__ __forceinline__ void bulk_load(uint32_t smem_dst, const void* gsrc, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_dst), "l"(gsrc), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t f32_order_key(float x) {
    const uint32_t u = __float_as_uint(x);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float f32_from_order_key(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// ---- work distribution -------------------------------------------------------------------------------------------
// A STEP is one key-block pair of one 128-query tile (16 MMAs, one pass of the epilogue); tile m of a sequence has
// steps(m) = ceil(visible key blocks / 2) of them.  All steps, in (sequence, tile, pair) order, are cut into gridDim.x
// contiguous ranges of equal length (+-1): every CTA does the same amount of work whatever the causal triangle looks like
// (items of a whole 32-block chunk dealt round-robin left the SMs idle 5 % of the launch, ncu sm active vs elapsed), and
// a CTA reloads the query tile only when its range crosses into the next tile.  A pair-step produces the complete maxima of
// its (2 query blocks x 2 key blocks), so cutting a tile's key range between CTAs needs no reduction.
// An ITEM is what the three roles hand to each other: up to 16 consecutive steps of one tile inside one 32-block chunk.
struct Item {
    int b, m, c;          // sequence, 128-query tile, 32-key-block chunk
    int pr0, pr1;         // pairs [pr0, pr1) of the chunk
    int nk;               // key blocks of the chunk the tile can see (1 .. PF_CHUNK)
    bool new_tile;        // first item of this (b, m) in this CTA: the query tile has to be loaded
};
struct ItemWalk {
    int b, m, p, left, steps_m;
    bool fresh;
    // steps of tile m: ceil(n_vis / 2), n_vis = qb_start + (last query block of the tile) + 1
    static __device__ __forceinline__ int steps_of(const PrefillScoreArgs& a, int m) {
        return (a.qb_start + min(2 * m + 1, a.n_qb - 1) + 2) >> 1;
    }
    // steps of tiles 0 .. m-1 (m <= n_qt - 1: all of them have both query blocks): sum of (m' + h), h = (qb_start + 3) / 2
    static __device__ __forceinline__ int64_t steps_before(const PrefillScoreArgs& a, int m) {
        return (int64_t)m * (m - 1) / 2 + (int64_t)m * ((a.qb_start + 3) >> 1);
    }
    __device__ __forceinline__ void init(const PrefillScoreArgs& a) {
        const int64_t lo = a.total_steps * blockIdx.x / gridDim.x, hi = a.total_steps * (blockIdx.x + 1) / gridDim.x;
        left = (int)(hi - lo);
        b = (int)(lo / a.steps_per_seq);
        const int64_t r = lo - (int64_t)b * a.steps_per_seq;
        int m_lo = 0, m_hi = a.n_qt - 1;                     // largest m with steps_before(m) <= r
        while (m_lo < m_hi) {
            const int mid = (m_lo + m_hi + 1) >> 1;
            if (steps_before(a, mid) <= r) m_lo = mid; else m_hi = mid - 1;
        }
        m = m_lo;
        p = (int)(r - steps_before(a, m));
        steps_m = steps_of(a, m);
        fresh = true;
    }
    __device__ __forceinline__ bool next(const PrefillScoreArgs& a, Item& it) {
        if (left <= 0) return false;
        constexpr int PPC = PF_CHUNK / 2;                     // pairs per chunk
        it.b = b; it.m = m; it.c = p / PPC; it.pr0 = p - it.c * PPC;
        const int n = min(min(PPC - it.pr0, steps_m - p), left);
        it.pr1 = it.pr0 + n;
        it.nk = min(PF_CHUNK, a.qb_start + min(2 * m + 1, a.n_qb - 1) + 1 - it.c * PF_CHUNK);
        it.new_tile = fresh;
        fresh = false;
        p += n; left -= n;
        if (p == steps_m) {
            p = 0; fresh = true;
            if (++m == a.n_qt) { m = 0; ++b; }
            steps_m = steps_of(a, m);
        }
        return true;
    }
};

// ring position of an accumulator: slot and the parity of its use
struct AccPos {
    int slot, par;
    __device__ __forceinline__ void next(int n) {
        if (++slot == n) { slot = 0; par ^= 1; }
    }
};

template <int HB, int KIND>
__global__ void __launch_bounds__((PfCfg<HB, KIND>::THREADS), 1) score_prefill_kernel(const __grid_constant__ CUtensorMap tm_q,
                                                                      const __grid_constant__ CUtensorMap tm_k,
                                                                      const PrefillScoreArgs a) {
    using Cfg = PfCfg<HB, KIND>;
    constexpr bool F8 = Cfg::F8, MX4 = Cfg::MX4;
    constexpr int PF_THREADS = Cfg::THREADS;
    constexpr int PF_KSTAGES = Cfg::KSTAGES, NACC = Cfg::NACC;
    constexpr uint32_t K_TILE_BYTES = Cfg::K_STAGE_BYTES, Q_TILE_BYTES = Cfg::Q_TILE_BYTES;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* smem = smem_raw + (smem_base - smem_u32(smem_raw));
    const uint32_t q_smem = smem_base;                               // the query tile
    const uint32_t k_smem = smem_base + Q_TILE_BYTES;                // the key ring
    unsigned char* misc = smem + Cfg::SMEM_TILES;
    const uint32_t misc_u32 = smem_base + Cfg::SMEM_TILES;
    // barriers (8 bytes each)
    const uint32_t bar_q_full = misc_u32 + 0;
    const uint32_t bar_q_empty = misc_u32 + 8;
    const uint32_t bar_k_full = misc_u32 + 16;     // [<= 8]
    const uint32_t bar_k_empty = misc_u32 + 80;    // [<= 8]
    const uint32_t bar_t_full = misc_u32 + 144;    // [<= 4]
    const uint32_t bar_t_empty = misc_u32 + 176;   // [<= 4]
    static_assert(PF_KSTAGES <= 8 && NACC <= 4, "barrier layout");
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(misc + 208);
    uint32_t* s_max = reinterpret_cast<uint32_t*>(misc + 224);       // [CHUNK][4 quarters][2 query blocks]
    const uint32_t bar_sfq_full = misc_u32 + 1280;                   // MX4: the scale words are in tensor memory
    const uint32_t bar_sfk_full = misc_u32 + 1288;                   // [<= 8]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        mbar_init(bar_q_full, 1);
        mbar_init(bar_q_empty, 1);
        for (int i = 0; i < PF_KSTAGES; ++i) {
            mbar_init(bar_k_full + 8 * i, 1);
            mbar_init(bar_k_empty + 8 * i, 1);
        }
        for (int i = 0; i < NACC; ++i) {
            mbar_init(bar_t_full + 8 * i, 1);
            mbar_init(bar_t_empty + 8 * i, PF_EPI_WARPS);
        }
        if constexpr (MX4) {
            mbar_init(bar_sfq_full, Cfg::SF_WARPS);
            for (int i = 0; i < PF_KSTAGES; ++i) mbar_init(bar_sfk_full + 8 * i, Cfg::SF_WARPS);
        }
        mbar_fence_init();
    }
    for (int e = threadIdx.x; e < PF_CHUNK * 4 * 2; e += PF_THREADS) s_max[e] = 0u;
    if (warp == 0) tmem_alloc(misc_u32 + 208, 512);
    if (warp == PF_EPI_WARPS && lane == 0) {
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tbase = *tmem_slot;
    pdl_wait();
    pdl_launch_dependents();

    if (warp >= PF_EPI_WARPS) {
    if constexpr (MX4) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");      // warpgroups 2, 3 (producer, issuer, scale movers)
    if (warp == PF_EPI_WARPS) {
        // ================================ TMA producer: the key ring ================================
        if (lane == 0) {
            int n_tile = 0, kp = 0;
            ItemWalk walk;
            walk.init(a);
            Item it;
            while (walk.next(a, it)) {
                const int b = it.b, c = it.c;
                if (it.new_tile) {                             // (n_tile counts the query tiles this CTA has loaded)
                    mbar_wait(bar_q_empty, (n_tile & 1) ^ 1);  // the previous tile's MMAs have completed
                    if constexpr (MX4) {
                        // codes: two 64-token tiles of the query cache (dims: 128 B, 64 rows, tiles, planes); scale rows: one
                        // bulk copy per tile that exists (a tile past the chunk holds no queries: its rows are masked)
                        const int t0 = 2 * it.m, nt = min(2, a.q_tiles - t0);
                        constexpr uint32_t SC = 64 * Cfg::NG, TB = 64 * (Cfg::PLANES * 128 + Cfg::NG);
                        mbar_arrive_expect_tx(bar_q_full, Cfg::Q_CODE_BYTES + nt * SC);
                        tma_load_4d(q_smem, &tm_q, bar_q_full, 0, 0, b * a.q_tiles + t0, 0);
                        for (int i = 0; i < nt; ++i)
                            bulk_load(q_smem + Cfg::Q_CODE_BYTES + i * SC,
                                      a.q_cache + ((int64_t)b * a.q_tiles + t0 + i) * TB + 64 * Cfg::PLANES * 128, SC, bar_q_full);
                    } else {
                        mbar_arrive_expect_tx(bar_q_full, Q_TILE_BYTES);
                        tma_load_4d(q_smem, &tm_q, bar_q_full, 0, it.m * PF_M, 0, b);
                    }
                    ++n_tile;
                }
                // (kp counts ring slots: one per pair, or one per (pair, head) at HB = 256)
                for (int pr = it.pr0; pr < it.pr1; ++pr)
                    for (int hh = 0; hh < (Cfg::PER_HEAD ? PF_H : 1); ++hh, ++kp) {
                        const int s = kp % PF_KSTAGES;
                        mbar_wait(bar_k_empty + 8 * s, ((kp / PF_KSTAGES) & 1) ^ 1);
                        if constexpr (MX4) {
                            const int t0 = c * PF_CHUNK + 2 * pr, nt = min(2, a.k_tiles - t0);
                            constexpr uint32_t SC = 64 * Cfg::NG, TB = 64 * (Cfg::PLANES * 128 + Cfg::NG);
                            mbar_arrive_expect_tx(bar_k_full + 8 * s, Cfg::K_CODE_BYTES + nt * SC);
                            // (a pair that overhangs the sequence reads the next sequence's first tile, or zeros past the
                            // cache: its second block is never used)
                            tma_load_4d(k_smem + s * K_TILE_BYTES, &tm_k, bar_k_full + 8 * s, 0, 0, b * a.k_tiles + t0, 0);
                            for (int i = 0; i < nt; ++i)
                                bulk_load(k_smem + s * K_TILE_BYTES + Cfg::K_CODE_BYTES + i * SC,
                                          a.k_cache + ((int64_t)b * a.k_tiles + t0 + i) * TB + 64 * Cfg::PLANES * 128, SC,
                                          bar_k_full + 8 * s);
                        } else {
                        mbar_arrive_expect_tx(bar_k_full + 8 * s, K_TILE_BYTES);
                        // a pair that overhangs the cache is zero-filled by TMA; its second block is never used
                        tma_load_4d(k_smem + s * K_TILE_BYTES, &tm_k, bar_k_full + 8 * s, 0, (c * PF_CHUNK + 2 * pr) * 64,
                                    hh * Cfg::HEAD_PLANES, b);
                        }
                        PF_STAMP(0, kp);
                    }
            }
        }
#ifdef SPOT_TRACE
        if (lane == 1 && a.trace && blockIdx.x == 5) {          // observer: when does each key slot actually arrive?
            int kp = 0;
            ItemWalk walk;
            walk.init(a);
            Item it;
            while (walk.next(a, it)) {
                for (int pr = it.pr0; pr < it.pr1; ++pr)
                    for (int hh = 0; hh < (Cfg::PER_HEAD ? PF_H : 1); ++hh, ++kp) {
                        const int s = kp % PF_KSTAGES;
                        mbar_wait(bar_k_full + 8 * s, (kp / PF_KSTAGES) & 1);
                        PF_STAMP(1, kp);
                    }
            }
        }
#endif
    } else if (warp == PF_EPI_WARPS + 1) {
        // ================================ MMA issuer ================================
        // The whole warp runs this loop converged; one elected lane issues (tc100.cuh, umma_*_elect).
        {
            constexpr uint32_t idesc = MX4 ? umma_idesc_mxf4(PF_M, PF_N) : F8 ? umma_idesc_e4m3(PF_M, PF_N) : umma_idesc_bf16(PF_M, PF_N);
            int n_tile = 0, kp = 0, acc = 0;
            AccPos ap{0, 0};
            const uint64_t qd = umma_desc_sw128(q_smem);
            ItemWalk walk;
            walk.init(a);
            Item it;
            while (walk.next(a, it)) {
                if (it.new_tile) {
                    // every MMA issued so far read the previous query tile: when they have completed, its buffer is free
                    if (n_tile > 0) umma_commit_elect(bar_q_empty);
                    mbar_wait(bar_q_full, n_tile & 1);         // this tile's queries have landed
                    if constexpr (MX4) mbar_wait(bar_sfq_full, n_tile & 1);   // ... and their scale words sit in tensor memory
                    tc_fence_after();
                    ++n_tile;
                }
                for (int pr = it.pr0; pr < it.pr1; ++pr) {
                    int s = 0;
                    uint64_t kd = 0;                           // descriptor of the slot's first byte
                    if constexpr (!Cfg::PER_HEAD) {
                        s = kp % PF_KSTAGES;
                        mbar_wait(bar_k_full + 8 * s, (kp / PF_KSTAGES) & 1);
                        if constexpr (MX4) mbar_wait(bar_sfk_full + 8 * s, (kp / PF_KSTAGES) & 1);
                        kd = umma_desc_sw128(k_smem + s * K_TILE_BYTES);
                        ++kp;
                    }
#pragma unroll
                    for (int h = 0; h < PF_H; ++h, ++acc) {
                        if constexpr (Cfg::PER_HEAD) {
                            s = kp % PF_KSTAGES;
                            mbar_wait(bar_k_full + 8 * s, (kp / PF_KSTAGES) & 1);
                            kd = umma_desc_sw128(k_smem + s * K_TILE_BYTES);
                            ++kp;
                        }
                        mbar_wait(bar_t_empty + 8 * ap.slot, ap.par ^ 1);
                        if (lane == 0) PF_STAMP(2, acc);
                        tc_fence_after();
                        const uint32_t d_tmem = tbase + ap.slot * PF_N;
#pragma unroll
                        for (int ks = 0; ks < Cfg::KSTEPS; ++ks) {
                            // the address field of the descriptor is (byte address >> 4): add the k-step's offset to it
                            const uint64_t bd = kd + (uint64_t)(Cfg::koff(Cfg::PER_HEAD ? 0 : h, ks) >> 4);
                            const uint64_t ad = qd + (uint64_t)(Cfg::koff(h, ks) >> 4);
                            if constexpr (MX4) {
                                // the k-step's two scales: groups g0, g0 + 1 of the token row = bytes g0 % 4, + 1 of scale word g0 / 4
                                const int g0 = (h * HB + ks * 32) / 16;
                                umma_mxf4_ss_elect(d_tmem, ad, bd, idesc | umma_idesc_sf_ids(g0 & 3, g0 & 3),
                                                   tbase + Cfg::SFQ_COL + 4 * (g0 >> 2),
                                                   tbase + Cfg::SFK_COL + 16 * s + 4 * (g0 >> 2), ks > 0);
                            } else if constexpr (F8) umma_f8_ss_elect(d_tmem, ad, bd, idesc, ks > 0);
                            else umma_bf16_ss_elect(d_tmem, ad, bd, idesc, ks > 0);
                        }
                        umma_commit_elect(bar_t_full + 8 * ap.slot);      // this head's accumulator is ready for the epilogue
                        if (lane == 0) PF_STAMP(3, acc);
                        if constexpr (Cfg::PER_HEAD) umma_commit_elect(bar_k_empty + 8 * s);
                        ap.next(NACC);
                    }
                    if constexpr (!Cfg::PER_HEAD) umma_commit_elect(bar_k_empty + 8 * s);   // slot free once these MMAs have read it
                }
            }
        }
    } else if (warp < PF_EPI_WARPS + 2 + Cfg::SF_WARPS) {
        // ================================ MX4: scale words into tensor memory (warps 10 .. 13) ================================
        // Warp w serves TMEM lane quarter w % 4 (the MMA wants the same words in all four).  A slot's scale bytes lie behind
        // its codes as [128 rows][NG]; word wd of row r goes to column 4 wd + r / 32 of the slot's block, lane r % 32.
        if constexpr (MX4) {
            constexpr int NW = Cfg::NG / 4;                  // 32-bit scale words per row: 2 (d_idx 64) / 4 (d_idx 128)
            const uint32_t lane_base = tbase + ((uint32_t)((warp & 3) * 32) << 16);
            auto move = [&](uint32_t sf_smem, uint32_t col, uint32_t bar) {
                uint32_t r[4 * NW];
#pragma unroll
                for (int wd = 0; wd < NW; ++wd)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r[4 * wd + j])
                                     : "r"(sf_smem + (uint32_t)((lane + 32 * j) * Cfg::NG + 4 * wd)));
#pragma unroll
                for (int wd = 0; wd < NW; ++wd) tmem_st4u(lane_base + col + 4 * wd, r + 4 * wd);
                tmem_st_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar);
            };
            int n_tile = 0, kp = 0;
            ItemWalk walk;
            walk.init(a);
            Item it;
            while (walk.next(a, it)) {
                if (it.new_tile) {
                    mbar_wait(bar_q_full, n_tile & 1);
                    move(q_smem + Cfg::Q_CODE_BYTES, Cfg::SFQ_COL, bar_sfq_full);
                    ++n_tile;
                }
                for (int pr = it.pr0; pr < it.pr1; ++pr, ++kp) {
                    const int s = kp % PF_KSTAGES;
                    mbar_wait(bar_k_full + 8 * s, (kp / PF_KSTAGES) & 1);
                    move(k_smem + s * K_TILE_BYTES + Cfg::K_CODE_BYTES, Cfg::SFK_COL + 16 * s, bar_sfk_full + 8 * s);
                }
            }
        }
    }
    } else {
        if constexpr (MX4) asm volatile("setmaxnreg.inc.sync.aligned.u32 192;");  // warpgroups 0, 1
        // ================================ epilogue (warps 0 .. 7) ================================
        // Warp w owns TMEM lanes 32 (w & 3) .. +31 (one query per lane) and the 64 accumulator columns of key block (w >> 2)
        // of the pair.  TMEM reads and the fp32 arithmetic overlap: a warp keeps one 32-column tcgen05.ld in flight while it
        // works on the previous one (wait::ld, issue the next load into the other buffer, compute; tcgen05.wait::ld waits for
        // every outstanding load, hence this order).
        constexpr int EC = PF_N / (PF_EPI_WARPS / 4);        // accumulator columns per warp: 64
        constexpr int NSUB = EC / 32;                        // 32-column loads per head
        constexpr int NU = PF_H * NSUB;                      // loads per key-block pair (even)
        const int lq = warp & 3, ch = warp >> 2;
        const int col0 = ch * EC;                 // first accumulator column of this warp
        const int kb_in_pair = col0 >> 6;         // which key block of the pair
        const int c_in_blk = col0 & 63;           // first key of the warp inside that block
        const int row = lq * 32 + lane;           // query row of the tile = TMEM lane
        const int qbl = lq >> 1;                  // which of the tile's two query blocks
        const uint32_t t_row = tbase + ((uint32_t)(lq * 32) << 16);
        const uint32_t t_lane = t_row + col0;
        int pc = 0;
        AccPos ap{0, 0};                          // the accumulator whose load is in flight / comes next
        ItemWalk walk;
        walk.init(a);
        Item it;
        while (walk.next(a, it)) {
            const int b = it.b, c = it.c, m = it.m, nk = it.nk;
            const int q_local = m * PF_M + row;                 // query index inside the chunk of Tq queries
            const bool q_exists = q_local < a.Tq;
            float4 wv = make_float4(0.f, 0.f, 0.f, 0.f);
            if (q_exists) wv = *reinterpret_cast<const float4*>(a.w + ((int64_t)b * a.Tq + q_local) * PF_H);
            const float wh0 = 0.5f * wv.x, wh1 = 0.5f * wv.y;   // heads 0-1: (w/2)(d + |d|)
            const int qb_abs = a.qb_start + 2 * m + qbl;        // this row's (absolute) query block = its diagonal
            const int q_in_blk = row & 63;
            float buf[2][32];
            mbar_wait(bar_t_full + 8 * ap.slot, ap.par);
            tc_fence_after();
            tmem_ld32(t_lane + ap.slot * PF_N, buf[0]);
            for (int pr = it.pr0; pr < it.pr1; ++pr, ++pc) {
                float S[EC];
#pragma unroll
                for (int u = 0; u < NU; ++u) {
                    const int h = u / NSUB, sb = u % NSUB;
                    tmem_ld_wait32(buf[u & 1]);
                    if (sb == 0 && warp == 0 && lane == 0) PF_STAMP(4, pc * 4 + h);
                    if (sb == NSUB - 1) {                       // head h fully read: hand its accumulator back
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(bar_t_empty + 8 * ap.slot);
                        if (warp == 0 && lane == 0) PF_STAMP(5, pc * 4 + h);
                        ap.next(NACC);
                    }
                    if (u + 1 < NU || pr + 1 < it.pr1) {
                        const int sb1 = (u + 1) % NSUB;
                        if (sb1 == 0) {                         // a new accumulator
                            mbar_wait(bar_t_full + 8 * ap.slot, ap.par);
                            tc_fence_after();
                        }
                        tmem_ld32(t_lane + ap.slot * PF_N + sb1 * 32, buf[(u + 1) & 1]);
                    }
                    const float (&dd)[32] = buf[u & 1];
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        float& s0 = S[sb * 32 + i];
                        float& s1 = S[sb * 32 + i + 1];
                        const float d0 = dd[i], d1 = dd[i + 1];
                        if (h == 0) {
                            fmul2(s0, s1, d0 + fabsf(d0), d1 + fabsf(d1), wh0);
                        } else if (h == 1) {
                            ffma2(s0, s1, d0 + fabsf(d0), d1 + fabsf(d1), wh1, s0, s1);
                        } else {
                            ffma2(s0, s1, fmaxf(d0, 0.f), fmaxf(d1, 0.f), h == 2 ? wv.z : wv.w, s0, s1);
                        }
                    }
                }
                const int kb = 2 * pr + kb_in_pair;             // this warp's key block of the pair
                const int j = c * PF_CHUNK + kb;
                if (j == qb_abs) {
                    // causal mask inside the diagonal tile: key t of the block is visible iff t <= q
#pragma unroll
                    for (int i = 0; i < EC; ++i)
                        if (c_in_blk + i > q_in_blk) S[i] = -INFINITY;
                }
                const bool live = kb < nk && j <= qb_abs && q_exists;   // warp-uniform: Tq is a multiple of 64, a warp's rows share a block
                if (a.row_blk) {
                    // rows form: this lane's query against the 64 keys of block j (masked keys are -inf: the diagonal block
                    // keeps at least key t = q0 for every row)
                    if (live) {
                        float q4m[4];
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) {
                            float mx = -INFINITY;
#pragma unroll
                            for (int i = 0; i < 16; i += 2) mx = fmax3(mx, S[q4 * 16 + i], S[q4 * 16 + i + 1]);
                            q4m[q4] = mx;
                        }
                        const float mrow = fmaxf(fmaxf(q4m[0], q4m[1]), fmaxf(q4m[2], q4m[3]));
                        float l0 = 0.f, l1 = 0.f;
#pragma unroll
                        for (int i = 0; i < EC; i += 2) {
                            l0 += fast_exp2((S[i] - mrow) * 1.4426950408889634f);
                            l1 += fast_exp2((S[i + 1] - mrow) * 1.4426950408889634f);
                        }
                        a.row_part[(int64_t)j * a.Tq + q_local] = make_float2(mrow, l0 + l1);
                        float* dst = a.row_blk + (int64_t)q_local * a.row_stride;
                        if (a.row_blk_tokens == 16) {
                            *reinterpret_cast<float4*>(dst + j * 4) = make_float4(q4m[0], q4m[1], q4m[2], q4m[3]);
                        } else if (a.row_blk_tokens == 32) {
                            *reinterpret_cast<float2*>(dst + j * 2) = make_float2(fmaxf(q4m[0], q4m[1]), fmaxf(q4m[2], q4m[3]));
                        } else {
                            dst[j] = mrow;
                        }
                    }
                } else if (!a.fine) {
                    float mx = -INFINITY;
#pragma unroll
                    for (int i = 0; i < EC; i += 2) mx = fmax3(mx, S[i], S[i + 1]);
                    if (live) {
                        const uint32_t key = __reduce_max_sync(0xffffffffu, f32_order_key(mx));
                        if (lane == 0) atomicMax(&s_max[(kb * 4) * 2 + qbl], key);
                    }
                } else {
                    // 16-token blocks (f3): one maximum per quarter of the 64-key block
#pragma unroll
                    for (int q4 = 0; q4 < EC / 16; ++q4) {
                        float mx = -INFINITY;
#pragma unroll
                        for (int i = 0; i < 16; i += 2) mx = fmax3(mx, S[q4 * 16 + i], S[q4 * 16 + i + 1]);
                        if (live) {
                            const uint32_t key = __reduce_max_sync(0xffffffffu, f32_order_key(mx));
                            if (lane == 0) atomicMax(&s_max[(kb * 4 + (c_in_blk >> 4) + q4) * 2 + qbl], key);
                        }
                    }
                }
            }
            if (a.row_blk) continue;                             // rows form: everything went out per step
            // item done: all epilogue warps meet, then the tile maxima go out and the buffer is re-armed
            asm volatile("bar.sync 1, %0;" :: "n"(PF_EPI_WARPS * 32) : "memory");
            const int nq4 = a.fine ? 4 : 1;
            const int kb_lo = 2 * it.pr0, kb_n = min(2 * it.pr1, nk) - kb_lo;      // the key blocks this item has scored
            for (int e = threadIdx.x; e < kb_n * nq4 * 2; e += PF_EPI_WARPS * 32) {
                const int qq = e & 1, q4 = (e >> 1) % nq4, kb = kb_lo + (e >> 1) / nq4;
                const int qblk = 2 * m + qq;
                const int j = c * PF_CHUNK + kb;
                const int slot = (kb * 4 + q4) * 2 + qq;
                const uint32_t key = s_max[slot];
                s_max[slot] = 0u;
                if (qblk < a.n_qb && j <= a.qb_start + qblk)
                    a.scores[((int64_t)b * a.n_qb + qblk) * a.nb_stride + j * nq4 + q4] = f32_from_order_key(key);
            }
            asm volatile("bar.sync 1, %0;" :: "n"(PF_EPI_WARPS * 32) : "memory");   // re-armed before the next item's maxima
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tbase, 512);
}

}  // namespace

// ---- host ---------------------------------------------------------------------------------------------------
bool encode_tmap_bf16_sw128(CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                            const uint64_t* strides_bytes, const uint32_t* box) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                 const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                 CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess || !p ||
            qres != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return false;
        }
        fn = reinterpret_cast<EncodeFn>(p);
    }
    cuuint64_t gdim[5], gstr[4];
    cuuint32_t bx[5], es[5];
    for (int i = 0; i < rank; ++i) { gdim[i] = dims[i]; bx[i] = box[i]; es[i] = 1; }
    for (int i = 0; i + 1 < rank; ++i) gstr[i] = strides_bytes[i];
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), gdim, gstr, bx, es,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// scores: fp32 [B * Tq/64][nb_stride]; entry (row, j) is written for every key block j the row's query block can see
struct PrefillRowsOut { float* blk_scores; int stride; float2* part; };

template <int HB, int KIND>
static spot_status score_prefill_d(const spot_select_params* p, float* scores, int nb_stride, cudaStream_t s,
                                   const PrefillRowsOut* rows = nullptr) {
    using Cfg = PfCfg<HB, KIND>;
    constexpr int PF_D = 64;                                        // plane width in BF16 pairs-of-bytes (128 bytes)
    constexpr int PLANES = Cfg::PLANES;
    PrefillScoreArgs a;
    a.w = p->w; a.scores = scores; a.nb_stride = nb_stride;
    a.B = p->B; a.Tq = p->Tq; a.n_qb = p->Tq / 64; a.n_qt = (a.n_qb + 1) / 2;
    a.qb_start = p->q_start / 64;
    a.fine = p->blk == 16;
    a.row_blk = rows ? rows->blk_scores : nullptr;
    a.row_part = rows ? rows->part : nullptr;
    a.row_stride = rows ? rows->stride : 0;
    a.row_blk_tokens = p->blk;
#ifdef SPOT_TRACE
    a.trace = g_pf_trace;
#endif
    // steps (ItemWalk): tiles 0 .. n_qt-2 have m + h of them, h = (qb_start + 3) / 2; the last tile may hold one query block
    {
        const int64_t last = a.n_qt - 1, h = (a.qb_start + 3) >> 1;
        const int64_t last_qb = (2 * last + 1 < a.n_qb - 1) ? 2 * last + 1 : a.n_qb - 1;
        a.steps_per_seq = last * (last - 1) / 2 + last * h + ((a.qb_start + last_qb + 2) >> 1);
        a.total_steps = a.steps_per_seq * a.B;
    }
    const int64_t total = a.total_steps;
    if (total <= 0) return SPOT_ERR_INVALID_ARG;

    CUtensorMap tm_q, tm_k;
    const uint64_t row_bytes = (uint64_t)PLANES * 128;              // one token: PF_H heads x HB bytes = PLANES x 128 bytes
    a.q_cache = nullptr; a.k_cache = nullptr; a.q_tiles = a.k_tiles = 0;
    if constexpr (Cfg::MX4) {
        // both operands in the opaque MXFP4 layout: 64-token tiles of [64][row_bytes] code bytes + [64][NG] scale bytes.
        // The map walks the code rows: (128 bytes, 64 rows of a tile, tiles of the whole cache, planes); a box is two tiles
        // of every plane, which lands as [plane][128 rows][128 B] in shared memory
        if (p->Tq % 64 != 0 || p->cache_stride_tokens % 64 != 0) return SPOT_ERR_INVALID_ARG;
        const uint64_t tile_bytes = 64 * (row_bytes + Cfg::NG);
        a.q_cache = (const uint8_t*)p->sel_q; a.k_cache = (const uint8_t*)p->sel_k;
        a.q_tiles = p->Tq / 64; a.k_tiles = (int)(p->cache_stride_tokens / 64);
        const void* base[2] = {p->sel_q, p->sel_k};
        const int tiles[2] = {a.q_tiles, a.k_tiles};
        CUtensorMap* tm[2] = {&tm_q, &tm_k};
        for (int i = 0; i < 2; ++i) {
            const uint64_t dims[4] = {(uint64_t)PF_D, 64, (uint64_t)p->B * tiles[i], (uint64_t)PLANES};
            const uint64_t strides[3] = {row_bytes, tile_bytes, 128};
            const uint32_t box[4] = {(uint32_t)PF_D, 64u, 2u, (uint32_t)PLANES};
            if (!encode_tmap_bf16_sw128(tm[i], base[i], 4, dims, strides, box)) return SPOT_ERR_CUDA;
        }
    } else {
    {
        const uint64_t dims[4] = {(uint64_t)PF_D, (uint64_t)p->Tq, (uint64_t)PLANES, (uint64_t)p->B};
        const uint64_t strides[3] = {row_bytes, (uint64_t)PF_D * 2, (uint64_t)p->Tq * row_bytes};
        const uint32_t box[4] = {(uint32_t)PF_D, (uint32_t)PF_M, (uint32_t)PLANES, 1u};
        if (!encode_tmap_bf16_sw128(&tm_q, p->sel_q, 4, dims, strides, box)) return SPOT_ERR_CUDA;
    }
    {
        const uint64_t dims[4] = {(uint64_t)PF_D, (uint64_t)p->cache_stride_tokens, (uint64_t)PLANES, (uint64_t)p->B};
        const uint64_t strides[3] = {row_bytes, (uint64_t)PF_D * 2, (uint64_t)p->cache_stride_tokens * row_bytes};
        // a pair of key blocks: every head's planes, or (HB = 256) one head's two planes
        const uint32_t box[4] = {(uint32_t)PF_D, (uint32_t)PF_N, (uint32_t)Cfg::STAGE_PLANES, 1u};
        if (!encode_tmap_bf16_sw128(&tm_k, p->sel_k, 4, dims, strides, box)) return SPOT_ERR_CUDA;
    }
    }
    static unsigned long long smem_attr_done = 0;
    SPOT_CUDA_TRY(set_max_smem_once(score_prefill_kernel<HB, KIND>, (int)Cfg::SMEM_BYTES, smem_attr_done));
    const int grid = (int)(total < sm_count() ? total : sm_count());
    SPOT_CUDA_TRY(launch_pdl(score_prefill_kernel<HB, KIND>, dim3((unsigned)grid), dim3(Cfg::THREADS), (size_t)Cfg::SMEM_BYTES, s,
                             tm_q, tm_k, a));
    return SPOT_OK;
}

// q_fmt: SPOT_SELK_FP8_E4M3 -- queries AND keys are FP8-E4M3 bytes ([..][H][d], the FP8 cache layout); SPOT_SELK_MXFP4 --
// both are MXFP4 caches (the queries: a cache of Tq tokens per sequence); SPOT_SELK_BF16 -- both are BF16
spot_status score_prefill(const spot_select_params* p, float* scores, int nb_stride, int q_fmt, cudaStream_t s) {
    if (p->H_idx != PF_H) return SPOT_ERR_UNSUPPORTED;
    if (q_fmt == SPOT_SELK_FP8_E4M3) {
        if (p->d_idx == 64) return score_prefill_d<64, PF_F8>(p, scores, nb_stride, s);
        if (p->d_idx == 128) return score_prefill_d<128, PF_F8>(p, scores, nb_stride, s);
        return SPOT_ERR_UNSUPPORTED;
    }
    if (q_fmt == SPOT_SELK_MXFP4) {
        if (p->d_idx == 64) return score_prefill_d<32, PF_MX4>(p, scores, nb_stride, s);
        if (p->d_idx == 128) return score_prefill_d<64, PF_MX4>(p, scores, nb_stride, s);
        return SPOT_ERR_UNSUPPORTED;
    }
    if (p->fmt != SPOT_SELK_BF16) return SPOT_ERR_UNSUPPORTED;      // other quantised caches: dequantised by the caller (api.cu)
    if (p->d_idx == 64) return score_prefill_d<128, PF_BF16>(p, scores, nb_stride, s);
    if (p->d_idx == 128) return score_prefill_d<256, PF_BF16>(p, scores, nb_stride, s);
    return SPOT_ERR_UNSUPPORTED;
}

// f4 (train_kl.cu): the student's pass 1 on the same kernel in its rows form -- one sequence of L = whole 64-query blocks,
// BF16 selector queries / keys [L][4][d_idx]; blk_scores [L][stride] gets every query's block maxima, part [L / 64][L] the
// per-64-key (max, sum exp) pairs of its scores.  blk in {16, 32, 64}.
spot_status score_prefill_rows(const uint16_t* sel_q, const float* w, const uint16_t* sel_k, int L, int H_idx, int d_idx,
                               int blk, float* blk_scores, int stride, float2* part, cudaStream_t s) {
    if (H_idx != PF_H || L % 64 != 0 || (blk != 16 && blk != 32 && blk != 64)) return SPOT_ERR_UNSUPPORTED;
    spot_select_params p;
    memset(&p, 0, sizeof(p));
    p.sel_q = sel_q; p.w = w; p.sel_k = sel_k; p.fmt = SPOT_SELK_BF16; p.cache_stride_tokens = L;
    p.B = 1; p.Tq = L; p.H_idx = H_idx; p.d_idx = d_idx; p.q_start = 0; p.blk = blk; p.q_block = 64;
    const PrefillRowsOut rows{blk_scores, stride, part};
    if (d_idx == 64) return score_prefill_d<128, PF_BF16>(&p, nullptr, 0, s, &rows);
    if (d_idx == 128) return score_prefill_d<256, PF_BF16>(&p, nullptr, 0, s, &rows);
    return SPOT_ERR_UNSUPPORTED;
}

}  // namespace spot

#ifdef SPOT_TRACE
extern "C" void spot_debug_set_pf_trace(void* dev_buf) { spot::g_pf_trace = (long long*)dev_buf; }
#endif
