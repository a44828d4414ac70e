// Step a1, decode form -- stream the selector K-cache once and emit one score per 64-token block:
//   s[t] = sum_h w_h ReLU(q_h . k_{h,t}),   s_bar[b] = max_{t in b} s[t].
//
// HBM-bound: 512 B (BF16) or 136 B (4-bit) per token, 2 flop/B, no reuse.  What limits a kernel like this is the
// number of bytes it keeps in flight (6.5 TB/s x ~1.5 us of loaded latency = ~10 MB = ~70 KiB per SM), so the loads
// are taken off the warps' registers: one persistent CTA per SM owns a contiguous range of the flat (sequence, tile)
// list and a producer lane streams its 64-token tiles through a shared-memory ring with the bulk-copy engine --
//   BF16 cache : one cp.async.bulk.tensor (TMA) per tile, box [d 64][64 tokens][H*d/64 planes], 128-byte swizzle
//                (32 KiB per tile at 4 x 64), so that ldmatrix reads of 8 token rows are bank-conflict free;
//   4-bit cache: one cp.async.bulk per tile; the opaque layout keeps a tile's codes and scales contiguous (8704 B)
// -- 144..192 KiB in flight per SM, completion on mbarriers.  Consumer warps (each owning its share of the ring's stages) take the tiles round-robin; a tile
// is 16-token row groups fed to mma.sync m16n8k16 with the query in column 0 of the B fragment (the tensor pipe is
// idle otherwise, so the 7 wasted columns are free) and the reduction over d_idx happens inside the MMA instead of
// in shuffles.
//   BF16 cache : bf16 HMMA, products exact, fp32 accumulate.
//   4-bit cache: codes are unpacked to fp16 pairs in registers (INT4: magic-number OR + one HFMA2 per pair;
//                MXFP4: cvt.rn.f16x2.e2m1x2, one instruction per pair), multiplied against an fp16 copy of the
//                query (pre-scaled per head by a power of two so that the copy is exact for every element
//                within 2^-29 of the head's largest), and the group scale is applied to the 32-element partial
//                sum after the MMA (one FMUL per group instead of one per element).  The k index of each MMA is a
//                fixed permutation of the d_idx axis applied to both operands, chosen so that every lane's 16-byte
//                shared-memory load lands directly in fragment registers.
//   FP8 cache  : (f2) one cvt.rn.f16x2.e4m3x2 per pair, no scales, the same fp16 HMMA.
//   INT4 with BF16 group scales (f2, R39): the INT4 path with two scale bytes per group, scale -> fp32 is a shift.
//   MXINT8 cache (f2, R38): code bytes are offset-binary u = code + 128; one PRMT per pair drops each byte into the low
//                end of an fp16 (the subnormal u 2^-24, exact), the offset 128 sum x is taken on the query side as for
//                INT4, the E8M0 scale and 2^-6 go into the post-scale.
// With 16-token blocks (f3, blk == 16) a tile yields its four 16-token maxima instead of one.
#include "common.cuh"
#include "tc100.cuh"

#include <string.h>
#include <type_traits>

namespace spot {

namespace {

constexpr int SC_SMEM_BUDGET = 196 * 1024;     // ring bytes per CTA (one CTA per SM)


// four bytes of E2M1 pairs -> four fp16 pairs; the vector mov lets ptxas use F2FP's byte selectors (.B0-.B3),
// one instruction per pair and no shift/mask.
__device__ __forceinline__ void e2m1x8_to_f16x2x4(uint32_t w, uint32_t (&p)[4]) {
    asm("{ .reg .b8 b0, b1, b2, b3; mov.b32 {b0, b1, b2, b3}, %4;\n"
        "cvt.rn.f16x2.e2m1x2 %0, b0; cvt.rn.f16x2.e2m1x2 %1, b1;\n"
        "cvt.rn.f16x2.e2m1x2 %2, b2; cvt.rn.f16x2.e2m1x2 %3, b3; }"
        : "=r"(p[0]), "=r"(p[1]), "=r"(p[2]), "=r"(p[3]) : "r"(w));
}

// 8 codes (one 32-bit word) -> 4 fp16 pairs; pair pp = dims (2pp, 2pp+1) of the word.
template <int FMT>
__device__ __forceinline__ void unpack8(uint32_t w, uint32_t (&p)[4]) {
    if (FMT == SPOT_SELK_MXFP4) {
        e2m1x8_to_f16x2x4(w, p);
    } else {
        // u = q + 8 in each nibble, read as it stands: four bits in the low end of an fp16 are the SUBNORMAL u 2^-24
        // (exact, and the tensor cores take fp16 subnormals), the nibble at bit 4 is 16 u 2^-24 -- one LOP3 per pair, no
        // magic-number fix-up.  The factor 16 is taken out of the QUERY's copy of those dims (a power of two: exact), the
        // factor 2^-24 goes into the power-of-two post-scale, and the offset, sum_i 8 x_i over the group, is a constant of
        // the query, subtracted from the group's partial sum after the MMA (Q4Tile::stage_raw).  (Round 1 rebuilt q with
        // OR 0x6400 / HSUB2 / HFMA2: 9 instructions per 8 codes against 5; the INT4 kernel was ALU-bound.)
        const uint32_t w8 = w >> 8;
        p[0] = w & 0x000f000fu;
        p[1] = w & 0x00f000f0u;
        p[2] = w8 & 0x000f000fu;
        p[3] = w8 & 0x00f000f0u;
    }
}

// two adjacent E4M3 scale bytes -> fp32 (exact): cvt.rn.f16x2.e4m3x2, low byte -> low half
__device__ __forceinline__ void e4m3x2_to_f32x2(uint32_t two_bytes, float& lo, float& hi) {
    uint32_t h2;
    asm("{ .reg .b16 t; cvt.u16.u32 t, %1; cvt.rn.f16x2.e4m3x2 %0, t; }" : "=r"(h2) : "r"(two_bytes));
    const __half2 hh = *reinterpret_cast<const __half2*>(&h2);
    lo = __low2float(hh);
    hi = __high2float(hh);
}

template <int FMT>
__device__ __forceinline__ float scale_to_f32(uint32_t byte) {
    if (FMT == SPOT_SELK_MXFP4 || FMT == SPOT_SELK_MXINT8) {
        return byte ? __uint_as_float(byte << 23) : __uint_as_float(0x00400000u);
    } else {
        // E4M3 -> fp32 (exact): normal: 2^(E-7)(1+m/8); subnormal: m 2^-9
        uint32_t E = (byte >> 3) & 0xf, m = byte & 7;
        float nrm = __uint_as_float(((E + 120u) << 23) | (m << 20));
        float sub = (float)m * 0.001953125f;
        return E ? nrm : sub;
    }
}


__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t r;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}
// contiguous global -> shared bulk copy (bytes a multiple of 16), completion counted on an mbarrier
__device__ __forceinline__ void bulk_load(uint32_t smem_dst, const void* gsrc, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_dst), "l"(gsrc), "r"(bytes), "r"(bar) : "memory");
}

template <int H, int D_IDX, int FMT>
struct ScoreCfg {
    static constexpr int ROW = H * D_IDX;                      // elements per token
    static constexpr int CODE_BYTES = ROW / 32 * selk_code_bytes_per_group(FMT);      // grouped formats: per token
    static constexpr int SCALE_BYTES = ROW / 32 * selk_scale_bytes_per_group(FMT);
    static constexpr int TILE_BYTES = FMT == SPOT_SELK_BF16 ? 64 * ROW * 2
                                      : FMT == SPOT_SELK_FP8_E4M3 ? 64 * ROW : 64 * (CODE_BYTES + SCALE_BYTES);
    static constexpr bool SELF = FMT != SPOT_SELK_BF16;
    // BF16 (producer ring): few big tiles (32 / 64 KiB, 1024-byte aligned for the 128-byte swizzle) and a light
    // ldmatrix + HMMA body.  One producer lane feeds the ring; every stage belongs to ONE consumer warp (stage s ->
    // warp s % CONSUMERS, CONSUMERS == STAGES), so a warp meets the phases of a stage's barrier strictly in order --
    // with stages shared in rotation a warp could wait for phase k+1 of a barrier whose phase k (another warp's tile)
    // has not completed yet, and a parity wait cannot tell those apart.
    // 4-bit (self-serve ring): many small tiles (8.5 / 17 KiB) and an ALU-heavy unpack.  A single producer lane cannot
    // issue a copy per ~350 cycles, so every consumer warp owns PER_WARP stages and refills a stage itself as soon as
    // it has consumed it: no producer warp, no empty barriers.  The unpack's dependent chains want warps more than
    // ring depth: 12 warps x 2 stages beat 8 x 3 (MXFP4 20 -> 17 us); 16 warps x 3 half-tile stages were slower again.
    // FP8 (self-serve ring, split tiles): a 16 / 32 KiB tile would leave room for 6 / 3 warps only, so a stage holds
    // an 8 KiB slice (32 / 16 tokens) and a warp walks the SPLIT slices of its tile through its two stages, keeping
    // the running block maximum in registers.  (4 KiB slices x 4 stages per warp: no faster, 39.9 vs 38.0 us score + select.)
    // The 17 KiB 4-bit tiles of d_idx = 128 get the same treatment (12 warps instead of 6): a slice is 32 tokens' codes
    // plus their scale bytes, two bulk copies on one barrier.
    // (round 2, measured and not kept: 32-token slices with FOUR stages per warp for the 8.5 KiB tiles of d_idx = 64 --
    // MXFP4 scoring alone 24.4 vs 22.8 us at B = 4, 64.3 vs 57.7 us at B = 16: two copies and two barrier phases per tile
    // cost more issue slots than the deeper ring wins back)
    // MXINT8 (16.5 / 33 KiB tiles): slices of 8 KiB of codes + their scale bytes, as FP8.
    static constexpr int SPLIT = FMT == SPOT_SELK_FP8_E4M3 ? TILE_BYTES / 8192
                                 : FMT == SPOT_SELK_MXINT8 ? 64 * CODE_BYTES / 8192 : (SELF && TILE_BYTES > 12288 ? 2 : 1);
    static constexpr int STAGE_BYTES = SELF ? TILE_BYTES / SPLIT : (TILE_BYTES + 1023) / 1024 * 1024;
    static constexpr int STAGES_RAW = SC_SMEM_BUDGET / STAGE_BYTES;
    static constexpr int PER_WARP = SELF ? (STAGE_BYTES <= 4608 ? 4 : 2) : 1;
    static constexpr int SELF_MAX = (208 * 1024 / STAGE_BYTES) / (PER_WARP ? PER_WARP : 1);   // warps that fit
    static constexpr int CONSUMERS = SELF ? (SELF_MAX > 12 ? 12 : SELF_MAX) : (STAGES_RAW > 6 ? 6 : STAGES_RAW);
    static constexpr int STAGES = CONSUMERS * PER_WARP;
    static constexpr int THREADS = (CONSUMERS + (SELF ? 0 : 1)) * 32;
    static_assert(STAGES * STAGE_BYTES <= 208 * 1024, "ring geometry");
    // query slots: one per sequence when the batch has at most Q_SLOTS of them (staged once, at kernel start), else one
    // per consumer warp (restaged whenever the warp changes sequence)
    static constexpr int Q_SLOTS = 16;
    static constexpr int Q_SLOT_BYTES = ROW * 2 + 128;      // + post-scales, w, and (INT4) the group offsets
    static constexpr int Q16_BYTES = Q_SLOTS * Q_SLOT_BYTES;
    static_assert(CONSUMERS <= Q_SLOTS, "a slot per consumer warp");
    static constexpr int SMEM_BYTES = 256 + 1024 + STAGES * STAGE_BYTES + 2 * STAGES * 8 + Q16_BYTES + 64;
};

struct ScoreArgs {
    const uint16_t* sel_q;        // [B][H][d]
    const float* w;               // [B][H]
    const uint8_t* sel_k;         // 4-bit formats: the cache; BF16: unused (the tensor map carries the address)
    int64_t tiles_per_seq;        // 4-bit formats: cache_stride_tokens / 64
    const int32_t* seq_len;
    int max_len;                  // host-side bound of seq_len: device values are clamped to [0, max_len]
    int B;
    float* scores;
    int nb_stride;
    int fine;                     // blk == 16: four block maxima per 64-token tile (f3)
    int n_groups;                 // the batch is scored in this many groups of consecutive sequences (TileCursor)
    unsigned long long* tagged;   // pipelined step: block scores go out as {tag, fp32 bits} words, [B][nb_stride]
    uint32_t tag;                 //   (nullptr: plain fp32 into `scores`)
#ifdef SPOT_TRACE
    StepSync sync;
#endif
};

// seq_len[b] as the kernels use it: clamped to what the grid, the score rows and the cache were sized for
__device__ __forceinline__ int seq_len_of(const ScoreArgs& a, int b) { return min(max(a.seq_len[b], 0), a.max_len); }

// tiles of sequence b.  The kernel copies the (clamped) tile counts of the first SC_NB_CACHE sequences into shared memory
// once, in one coalesced load: the cursors below consult them on every change of sequence, and a chain of dependent
// global loads in front of the first tile request is what a short kernel cannot afford.
constexpr int SC_NB_CACHE = 64;
__device__ __forceinline__ int tiles_of(const ScoreArgs& a, int b) {
    extern __shared__ unsigned char smem_raw[];
    if (b < SC_NB_CACHE) return reinterpret_cast<const int*>(smem_raw)[b];
    return (seq_len_of(a, b) + 63) >> 6;
}

// Work assignment.  The batch is cut into n_groups groups of consecutive sequences (4, or B if smaller) and the whole grid
// walks them group by group -- so the block scores of group 0 are complete a quarter into the kernel, and the selection
// of its sequences (another kernel, resident beside this one) overlaps the scoring of the later groups.  Inside a group
// the CTAs split the flat (sequence, tile) list into equal CONTIGUOUS ranges, so a warp changes sequence (and reloads
// its query fragments: expensive for the quantised formats) about once per group, not once per tile.  Range c' of group
// g goes to CTA (c' + off_g) mod n with off_g the number of tiles in front of the group: with groups shorter than n tiles
// the non-empty ranges of consecutive groups land on consecutive CTAs instead of on the same few.
// The CTA's work list is the concatenation of its ranges; the cursor names a position in it.  The ranges (64-bit
// divisions) are worked out once per CTA into shared memory -- walking them costs a few integer instructions per tile,
// in kernels whose 4-bit forms are issue-bound.
constexpr int SC_MAX_GROUPS = 4;
struct CtaRange { int b0, t0, len; };             // first sequence, first tile of it, tiles in the range
// (thread g works out group g; 32-bit arithmetic -- a 64-bit division is a ~100-instruction dependent chain, and this
// sits in front of the first tile request: floor(rot T / n) = rot (T / n) + floor(rot (T % n) / n), all below 2^32 for
// n < 65536 CTAs and fewer than 2^32 / n tiles per group... the batch total is what must stay below 2^32 tiles)
__device__ __forceinline__ void cta_range_of_group(const ScoreArgs& a, int g, CtaRange* out) {
    const uint32_t n = gridDim.x;
    const int b0 = (int)((long long)g * a.B / a.n_groups), b1 = (int)((long long)(g + 1) * a.B / a.n_groups);
    uint32_t before = 0, T = 0;
    for (int bb = 0; bb < b0; ++bb) before += (uint32_t)tiles_of(a, bb);
    for (int bb = b0; bb < b1; ++bb) T += (uint32_t)tiles_of(a, bb);
    const uint32_t rot = (blockIdx.x + n - before % n) % n;          // which range of the group is this CTA's
    const uint32_t q = T / n, r = T - q * n;
    uint32_t i0 = rot * q + rot * r / n;
    const uint32_t i1 = (rot + 1) * q + (rot + 1) * r / n;
    out[g].len = (int)(i1 - i0);
    int b = b0;
    if (i1 > i0) {
        uint32_t nb = (uint32_t)tiles_of(a, b);
        while (i0 >= nb) { i0 -= nb; ++b; nb = (uint32_t)tiles_of(a, b); }
    }
    out[g].b0 = b;
    out[g].t0 = (int)i0;
}
struct TileCursor {
    int b, t, nb;                 // tile t of sequence b, which has nb tiles
    int left;                     // tiles of this CTA's range of group g at or after the cursor (<= 0: past the end)
    int g;
    // place the cursor `skip` tiles past the start of group gg's range, moving on to later groups as needed
    __device__ __forceinline__ void enter(const ScoreArgs& a, const CtaRange* rng, int gg, int skip) {
        g = gg;
        while (g < a.n_groups && skip >= rng[g].len) { skip -= rng[g].len; ++g; }
        if (g >= a.n_groups) { left = 0; return; }
        left = rng[g].len - skip;
        b = rng[g].b0; t = rng[g].t0 + skip; nb = tiles_of(a, b);
        while (t >= nb) { t -= nb; ++b; nb = tiles_of(a, b); }
    }
    __device__ __forceinline__ void first(const ScoreArgs& a, const CtaRange* rng) { enter(a, rng, 0, 0); }
    __device__ __forceinline__ void advance(const ScoreArgs& a, const CtaRange* rng, int n) {
        if (n < left) {
            left -= n; t += n;
            while (t >= nb) { t -= nb; ++b; nb = tiles_of(a, b); }
            return;
        }
        if (left > 0) enter(a, rng, g + 1, n - left);
    }
};

// Column 0 of the accumulators lives on lanes c == 0: the maximum over the 8 row lanes.
__device__ __forceinline__ float rows_max(float m, int lane) {
    if ((lane & 3) != 0) m = -INFINITY;
    m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 4));
    m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 8));
    m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 16));
    return m;
}
// One 16-token group (rows g and g + 8 of an MMA) has been scored.  Coarse (blk 64): fold it into the lane's running
// maximum, reduced over lanes once per tile.  Fine (blk 16, f3): reduce now and leave the group's maximum on lane 4 * grp.
__device__ __forceinline__ float group_update(float m, float sa, float sb, bool va, bool vb, int grp, int lane, bool fine) {
    float mi = va ? sa : -INFINITY;
    if (vb) mi = fmaxf(mi, sb);
    if (!fine) return fmaxf(m, mi);
    mi = rows_max(mi, lane);               // valid on lanes c == 0
    return lane == 4 * grp ? mi : m;
}

// One query row on its way to a shared-memory slot: the global loads are issued at the very start of the kernel (two
// DRAM round trips that would otherwise sit in front of the first tile), the conversion happens after the first tile
// requests are out.
struct QRaw { uint4 v[2]; float w; };

// ---- BF16 tile: planes [H * D_IDX / 64][64 tokens][128 B], 128-byte swizzle --------------------------------
template <int H, int D_IDX>
struct Bf16Tile {
    static constexpr int PPH = D_IDX / 64;       // planes per head
    static constexpr int NP = H * PPH;
    uint32_t qf[NP][4][2];
    float wh[H];

    // slot: ROW BF16 (the query as it is) + H floats (w)
    static __device__ __forceinline__ void load_raw(const ScoreArgs& a, int b, int lane, QRaw& r) {
        constexpr int ROW = H * D_IDX;
        static_assert(ROW / 8 <= 64, "two 16-byte chunks per lane");
        const uint4* src = reinterpret_cast<const uint4*>(a.sel_q + (int64_t)b * ROW);
#pragma unroll
        for (int i = 0; i < 2; ++i)
            if (i * 32 + lane < ROW / 8) r.v[i] = src[i * 32 + lane];
        r.w = lane < H ? a.w[(int64_t)b * H + lane] : 0.f;
    }
    static __device__ __forceinline__ void stage_raw(const QRaw& r, int lane, uint32_t slot) {
        constexpr int ROW = H * D_IDX;
        uint16_t* dst = reinterpret_cast<uint16_t*>(__cvta_shared_to_generic((size_t)slot));
#pragma unroll
        for (int i = 0; i < 2; ++i)
            if (i * 32 + lane < ROW / 8) reinterpret_cast<uint4*>(dst)[i * 32 + lane] = r.v[i];
        if (lane < H) reinterpret_cast<float*>(dst + ROW)[lane] = r.w;
        __syncwarp();
    }
    __device__ __forceinline__ void fetch(int lane, uint32_t slot) {
        constexpr int ROW = H * D_IDX;
        const int g = lane >> 2, c = lane & 3;
        const uint16_t* q = reinterpret_cast<const uint16_t*>(__cvta_shared_to_generic((size_t)slot));
#pragma unroll
        for (int pl = 0; pl < NP; ++pl)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                qf[pl][ks][0] = (g == 0) ? *reinterpret_cast<const uint32_t*>(q + pl * 64 + ks * 16 + 2 * c) : 0u;
                qf[pl][ks][1] = (g == 0) ? *reinterpret_cast<const uint32_t*>(q + pl * 64 + ks * 16 + 8 + 2 * c) : 0u;
            }
#pragma unroll
        for (int h = 0; h < H; ++h) wh[h] = reinterpret_cast<const float*>(q + ROW)[h];
    }

    // max over the tile's valid tokens of s[t]; valid on every lane after the final shuffles
    // (fine: lane 4 i, i < 4, returns the maximum over tokens [16 i, 16 i + 16) of the tile instead)
    __device__ __forceinline__ float tile_max(uint32_t st, int t0, int L, int lane, bool fine) const {
        const int g = lane >> 2, c = lane & 3, mi = lane >> 3, r8 = lane & 7;
        float m = -INFINITY;
#pragma unroll 1
        for (int rg = 0; rg < 4; ++rg) {
            const int row = rg * 16 + (mi & 1) * 8 + r8;
            const uint32_t rbase = st + row * 128;
            const int sw = row & 7;
            float sa = 0.f, sb = 0.f;
#pragma unroll
            for (int h = 0; h < H; ++h) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int sub = 0; sub < PPH; ++sub) {
                    const int pl = h * PPH + sub;
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks) {
                        uint32_t a0, a1, a2, a3;
                        ldmatrix_x4(a0, a1, a2, a3, rbase + pl * 8192 + (((2 * ks + (mi >> 1)) ^ sw) << 4));
                        mma_bf16_16816(acc, a0, a1, a2, a3, qf[pl][ks][0], qf[pl][ks][1]);
                    }
                }
                sa = fmaf(wh[h], fmaxf(acc[0], 0.f), sa);   // column 0, row g     (valid on lanes c == 0)
                sb = fmaf(wh[h], fmaxf(acc[2], 0.f), sb);   // column 0, row g + 8
            }
            const int ta = t0 + rg * 16 + g, tb = ta + 8;
            m = group_update(m, sa, sb, ta < L, tb < L, rg, lane, fine);
        }
        return fine ? m : rows_max(m, lane);
    }
};

// ---- 4-bit tile: [64][ROW/2] code bytes, then [64][ROW/32] scale bytes ------------------------------------
template <int H, int D_IDX, int FMT>
struct Q4Tile {
    static constexpr int ROW = H * D_IDX;
    static constexpr int CPT = ROW / 2;            // code bytes per token
    static constexpr int NG = ROW / 32;            // groups (= scale bytes) per token
    static constexpr int NQL = NG / 4;             // 64-byte "quad loads" per token: 4 groups, one per lane of a quad
    static constexpr int GPH = D_IDX / 32;         // groups per head (2 or 4)
    static constexpr bool IS_INT4 = FMT == SPOT_SELK_INT4_E4M3 || FMT == SPOT_SELK_INT4_BF16S;
    static constexpr int SB = selk_scale_bytes_per_group(FMT);   // scale bytes per group (2: BF16 scales, R39)
    static_assert(GPH == 2 || GPH == 4, "d_idx must be 64 or 128 for the 4-bit scoring kernels");
    static_assert(NG % 4 == 0, "H_idx * d_idx must be a multiple of 128");
    uint32_t qf[NQL][16];
    float wq[NQL], ps[NQL];
    float cq[NQL][2];                              // INT4: the offsets 8 sum x 2^-24 of this lane's two groups per quad load

    // slot: ROW halfs (the pre-scaled fp16 query) + H floats (power-of-two post-scales) + H floats (w)
    static __device__ __forceinline__ void load_raw(const ScoreArgs& a, int b, int lane, QRaw& r) {
        constexpr int EPL = ROW / 32;
        static_assert(EPL / 8 <= 2, "two 16-byte chunks per lane");
#pragma unroll
        for (int i = 0; i < EPL / 8; ++i)
            r.v[i] = *reinterpret_cast<const uint4*>(a.sel_q + (int64_t)b * ROW + lane * EPL + i * 8);
        r.w = lane < H ? a.w[(int64_t)b * H + lane] : 0.f;
    }
    static __device__ __forceinline__ void stage_raw(const QRaw& r, int lane, uint32_t q16_addr) {
        __half* q16 = reinterpret_cast<__half*>(__cvta_shared_to_generic((size_t)q16_addr));
        float* post = reinterpret_cast<float*>(q16 + ROW);
        // fp16 copy of q, pre-scaled per head by 2^sh so that the head's largest element lands in [2^14, 2^15).
        // One coalesced read of the whole query: lane l holds elements [EPL l, EPL l + EPL), 32 / H lanes per head.
        constexpr int EPL = ROW / 32, LPH = 32 / H;
        static_assert(EPL % 8 == 0 && LPH * EPL == D_IDX && (LPH & (LPH - 1)) == 0, "query staging geometry");
        __syncwarp();
        float v[EPL], mx = 0.f;
#pragma unroll
        for (int i = 0; i < EPL / 8; ++i) {
            const uint32_t wds[4] = {r.v[i].x, r.v[i].y, r.v[i].z, r.v[i].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) { v[i * 8 + 2 * j] = bf16lo(wds[j]); v[i * 8 + 2 * j + 1] = bf16hi(wds[j]); }
        }
#pragma unroll
        for (int i = 0; i < EPL; ++i) mx = fmaxf(mx, fabsf(v[i]));
#pragma unroll
        for (int o = LPH / 2; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        int sh = 0;
        if (mx > 0.f) sh = 14 - ilogbf(mx);
        sh = max(-100, min(100, sh));
        const float up = __uint_as_float((uint32_t)(127 + sh) << 23);
        if (IS_INT4) {
            // (see unpack8) dims 2, 3, 6, 7 of every 8 go in divided by 16; the group offset 8 sum x, times 2^-24
            float xs = 0.f;
#pragma unroll
            for (int i = 0; i < EPL; ++i) {
                const bool hi_nibble = (i & 2) != 0;              // EPL % 8 == 0: i % 8 is the dim inside its 8-code word
                const __half hq = __float2half_rn(v[i] * up * (hi_nibble ? 0.0625f : 1.0f));
                q16[lane * EPL + i] = hq;
                xs += __half2float(hq) * (hi_nibble ? 16.0f : 1.0f);
            }
            constexpr int LPG = 32 / EPL;                         // lanes per 32-element group
#pragma unroll
            for (int o = LPG / 2; o; o >>= 1) xs += __shfl_xor_sync(0xffffffffu, xs, o);
            if (lane % LPG == 0) post[2 * H + lane / LPG] = xs * (8.0f * 5.9604644775390625e-08f);
            if (lane % LPH == 0) post[lane / LPH] = __uint_as_float((uint32_t)(127 - sh + 24) << 23);
        } else {
#pragma unroll
            for (int i = 0; i < EPL; ++i) q16[lane * EPL + i] = __float2half_rn(v[i] * up);
            if (lane % LPH == 0) post[lane / LPH] = __uint_as_float((uint32_t)(127 - sh) << 23);
        }
        if (lane < H) post[H + lane] = r.w;
        __syncwarp();
    }
    __device__ __forceinline__ void fetch(int lane, uint32_t q16_addr) {
        const int g = lane >> 2, c = lane & 3;
        const __half* q16 = reinterpret_cast<const __half*>(__cvta_shared_to_generic((size_t)q16_addr));
        const float* post = reinterpret_cast<const float*>(q16 + ROW);
        // B fragments: column n of the MMA is the group held by quad-lane c == n; only lane (g == n, c == n) is non-zero
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
        // lanes c < 2 read columns 2c, 2c+1 = groups 4ql + 2c (+1); their head, weight and power-of-two post-scale
#pragma unroll
        for (int ql = 0; ql < NQL; ++ql) {
            const int head = (4 * ql + 2 * (c & 1)) / GPH;
            wq[ql] = post[H + head];
            ps[ql] = post[head];
            if (IS_INT4) {
                cq[ql][0] = post[2 * H + 4 * ql + 2 * (c & 1)];
                cq[ql][1] = post[2 * H + 4 * ql + 2 * (c & 1) + 1];
            }
        }
    }

    // maximum over the NIT * 16 tokens of a slice whose codes start at shared address st and whose scale bytes follow
    // them ([NIT*16][CPT] then [NIT*16][NG]); it0 = the slice's first 16-token group inside its tile (fine form)
    template <int NIT>
    __device__ __forceinline__ float part_max(uint32_t st, int t0, int L, int lane, bool fine, int it0) const {
        const int g = lane >> 2, c = lane & 3;
        float m = -INFINITY;
#pragma unroll 2
        for (int it = 0; it < NIT; ++it) {
            uint4 cd[NQL][2];
            uint32_t scw[2][NQL];
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const int tok = it * 16 + hf * 8 + g;
#pragma unroll
                for (int ql = 0; ql < NQL; ++ql) {
                    cd[ql][hf] = lds128(st + tok * CPT + ql * 64 + c * 16);
                    scw[hf][ql] = SB == 2 ? lds32(st + NIT * 16 * CPT + tok * NG * 2 + ql * 8 + 4 * (c & 1))   // this lane's two
                                          : lds32(st + NIT * 16 * CPT + tok * NG + ql * 4);
                }
            }
            float srow[2] = {0.f, 0.f};
#pragma unroll
            for (int ql = 0; ql < NQL; ++ql) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
                const uint32_t wa[4] = {cd[ql][0].x, cd[ql][0].y, cd[ql][0].z, cd[ql][0].w};
                const uint32_t wb[4] = {cd[ql][1].x, cd[ql][1].y, cd[ql][1].z, cd[ql][1].w};
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
                    const int gi = 2 * (c & 1);                        // first of this lane's two groups in the quad load
                    const uint32_t sw = scw[hf][ql];                   // scale bytes of groups 4ql .. 4ql+3
                    float s0, s1, d;
                    if (IS_INT4) {
                        if (SB == 2) { s0 = __uint_as_float(sw << 16); s1 = __uint_as_float(sw & 0xffff0000u); }   // BF16 bits
                        else e4m3x2_to_f32x2((sw >> (8 * gi)) & 0xffffu, s0, s1);
                        d = fmaf(acc[2 * hf] - cq[ql][0], s0, (acc[2 * hf + 1] - cq[ql][1]) * s1);
                    } else {
                        s0 = scale_to_f32<FMT>((sw >> (8 * gi)) & 0xffu);
                        s1 = scale_to_f32<FMT>((sw >> (8 * (gi + 1))) & 0xffu);
                        d = fmaf(acc[2 * hf], s0, acc[2 * hf + 1] * s1);
                    }
                    if (GPH == 4) d += __shfl_xor_sync(0xffffffffu, d, 1);   // the head's other two groups
                    d *= ps[ql];
                    float contrib = wq[ql] * fmaxf(d, 0.f);
                    if (GPH == 4 && (c & 1)) contrib = 0.f;           // counted once
                    srow[hf] += contrib;
                }
            }
            // heads are split over quad lanes 0 and 1
            const float sa = srow[0] + __shfl_xor_sync(0xffffffffu, srow[0], 1);
            const float sb = srow[1] + __shfl_xor_sync(0xffffffffu, srow[1], 1);
            const int ta = t0 + it * 16 + g, tbk = ta + 8;
            m = group_update(m, sa, sb, ta < L, tbk < L, it0 + it, lane, fine);
        }
        return fine ? m : rows_max(m, lane);
    }
};

// ---- MXINT8 tile (f2, R38): [tokens][ROW] offset-binary code bytes, then [tokens][ROW/32] E8M0 bytes ------------------
// The Q4 scheme with 32 code bytes per group: a quad load is 128 bytes of a token (four groups), stored as two 64-byte
// halves (quantize.cu: odd tokens keep them swapped), so that a lane's two 16-byte loads are bytes [0, 16) and [16, 32)
// of its group and the loads of two adjacent token rows fall into different banks.
template <int H, int D_IDX>
struct Q8Tile {
    static constexpr int ROW = H * D_IDX;
    static constexpr int CPT = ROW;                // code bytes per token
    static constexpr int NG = ROW / 32;            // groups (= scale bytes) per token
    static constexpr int NQL = NG / 4;             // 128-byte quad loads per token
    static constexpr int GPH = D_IDX / 32;
    static_assert(GPH == 2 || GPH == 4, "d_idx must be 64 or 128 for the MXINT8 scoring kernel");
    static_assert(NG % 4 == 0, "H_idx * d_idx must be a multiple of 128");
    uint32_t qf[NQL][16];
    float wq[NQL], ps[NQL];
    float cq[NQL][2];                              // the offsets 128 sum x 2^-24 of this lane's two groups per quad load

    static __device__ __forceinline__ void load_raw(const ScoreArgs& a, int b, int lane, QRaw& r) {
        constexpr int EPL = ROW / 32;
        static_assert(EPL / 8 <= 2, "two 16-byte chunks per lane");
#pragma unroll
        for (int i = 0; i < EPL / 8; ++i)
            r.v[i] = *reinterpret_cast<const uint4*>(a.sel_q + (int64_t)b * ROW + lane * EPL + i * 8);
        r.w = lane < H ? a.w[(int64_t)b * H + lane] : 0.f;
    }
    // slot: ROW halfs (the pre-scaled fp16 query) + H floats (power-of-two post-scales) + H floats (w) + NG floats (offsets)
    static __device__ __forceinline__ void stage_raw(const QRaw& r, int lane, uint32_t q16_addr) {
        __half* q16 = reinterpret_cast<__half*>(__cvta_shared_to_generic((size_t)q16_addr));
        float* post = reinterpret_cast<float*>(q16 + ROW);
        constexpr int EPL = ROW / 32, LPH = 32 / H;
        static_assert(EPL % 8 == 0 && LPH * EPL == D_IDX && (LPH & (LPH - 1)) == 0, "query staging geometry");
        __syncwarp();
        float v[EPL], mx = 0.f;
#pragma unroll
        for (int i = 0; i < EPL / 8; ++i) {
            const uint32_t wds[4] = {r.v[i].x, r.v[i].y, r.v[i].z, r.v[i].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) { v[i * 8 + 2 * j] = bf16lo(wds[j]); v[i * 8 + 2 * j + 1] = bf16hi(wds[j]); }
        }
#pragma unroll
        for (int i = 0; i < EPL; ++i) mx = fmaxf(mx, fabsf(v[i]));
#pragma unroll
        for (int o = LPH / 2; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        int sh = 0;
        if (mx > 0.f) sh = 14 - ilogbf(mx);
        sh = max(-100, min(100, sh));
        const float up = __uint_as_float((uint32_t)(127 + sh) << 23);
        float xs = 0.f;
#pragma unroll
        for (int i = 0; i < EPL; ++i) {
            const __half hq = __float2half_rn(v[i] * up);
            q16[lane * EPL + i] = hq;
            xs += __half2float(hq);
        }
        constexpr int LPG = 32 / EPL;                         // lanes per 32-element group
#pragma unroll
        for (int o = LPG / 2; o; o >>= 1) xs += __shfl_xor_sync(0xffffffffu, xs, o);
        if (lane % LPG == 0) post[2 * H + lane / LPG] = xs * (128.0f * 5.9604644775390625e-08f);
        // codes come in as u 2^-24 and mean code 2^-6: post-scale 2^(-sh + 24 - 6)
        if (lane % LPH == 0) post[lane / LPH] = __uint_as_float((uint32_t)(127 - sh + 18) << 23);
        if (lane < H) post[H + lane] = r.w;
        __syncwarp();
    }
    __device__ __forceinline__ void fetch(int lane, uint32_t q16_addr) {
        const int g = lane >> 2, c = lane & 3;
        const __half* q16 = reinterpret_cast<const __half*>(__cvta_shared_to_generic((size_t)q16_addr));
        const float* post = reinterpret_cast<const float*>(q16 + ROW);
        // B fragments: column n of the MMA is the group held by quad-lane c == n; only lane (g == n, c == n) is non-zero
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
#pragma unroll
        for (int ql = 0; ql < NQL; ++ql) {
            const int head = (4 * ql + 2 * (c & 1)) / GPH;
            wq[ql] = post[H + head];
            ps[ql] = post[head];
            cq[ql][0] = post[2 * H + 4 * ql + 2 * (c & 1)];
            cq[ql][1] = post[2 * H + 4 * ql + 2 * (c & 1) + 1];
        }
    }

    template <int NIT>
    __device__ __forceinline__ float part_max(uint32_t st, int t0, int L, int lane, bool fine, int it0) const {
        const int g = lane >> 2, c = lane & 3;
        const uint32_t first = (g & 1) ? 64u : 0u;            // where this token row keeps bytes [0, 16) of its groups
        float m = -INFINITY;
#pragma unroll 2
        for (int it = 0; it < NIT; ++it) {
            uint4 cd[NQL][2][2];
            uint32_t scw[2][NQL];
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                const int tok = it * 16 + hf * 8 + g;        // parity of tok == parity of g
#pragma unroll
                for (int ql = 0; ql < NQL; ++ql) {
                    cd[ql][hf][0] = lds128(st + tok * CPT + ql * 128 + first + c * 16);
                    cd[ql][hf][1] = lds128(st + tok * CPT + ql * 128 + (first ^ 64u) + c * 16);
                    scw[hf][ql] = lds32(st + NIT * 16 * CPT + tok * NG + ql * 4);
                }
            }
            float srow[2] = {0.f, 0.f};
#pragma unroll
            for (int ql = 0; ql < NQL; ++ql) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    const uint32_t wa[4] = {cd[ql][0][hh].x, cd[ql][0][hh].y, cd[ql][0][hh].z, cd[ql][0][hh].w};
                    const uint32_t wb[4] = {cd[ql][1][hh].x, cd[ql][1][hh].y, cd[ql][1][hh].z, cd[ql][1][hh].w};
#pragma unroll
                    for (int wd = 0; wd < 4; ++wd) {
                        // bytes (b0, b1) and (b2, b3) of the word as fp16 pairs 0x00b0, 0x00b1 | 0x00b2, 0x00b3
                        const uint32_t a0 = __byte_perm(wa[wd], 0u, 0x4140), a2 = __byte_perm(wa[wd], 0u, 0x4342);
                        const uint32_t a1 = __byte_perm(wb[wd], 0u, 0x4140), a3 = __byte_perm(wb[wd], 0u, 0x4342);
                        mma_f16_16816(acc, a0, a1, a2, a3, qf[ql][8 * hh + 2 * wd], qf[ql][8 * hh + 2 * wd + 1]);
                    }
                }
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int gi = 2 * (c & 1);
                    const uint32_t sw = scw[hf][ql];
                    const float s0 = scale_to_f32<SPOT_SELK_MXINT8>((sw >> (8 * gi)) & 0xffu);
                    const float s1 = scale_to_f32<SPOT_SELK_MXINT8>((sw >> (8 * (gi + 1))) & 0xffu);
                    float d = fmaf(acc[2 * hf] - cq[ql][0], s0, (acc[2 * hf + 1] - cq[ql][1]) * s1);
                    if (GPH == 4) d += __shfl_xor_sync(0xffffffffu, d, 1);
                    d *= ps[ql];
                    float contrib = wq[ql] * fmaxf(d, 0.f);
                    if (GPH == 4 && (c & 1)) contrib = 0.f;
                    srow[hf] += contrib;
                }
            }
            const float sa = srow[0] + __shfl_xor_sync(0xffffffffu, srow[0], 1);
            const float sb = srow[1] + __shfl_xor_sync(0xffffffffu, srow[1], 1);
            const int ta = t0 + it * 16 + g, tbk = ta + 8;
            m = group_update(m, sa, sb, ta < L, tbk < L, it0 + it, lane, fine);
        }
        return fine ? m : rows_max(m, lane);
    }
};

// ---- FP8-E4M3 tile (f2): [64 tokens][ROW] bytes, one byte per element, no scales ---------------------------
// Same scheme as the 4-bit tiles -- fp16 HMMA against the power-of-two pre-scaled fp16 query, the k index a fixed
// permutation so that a lane's 16-byte load lands in fragment registers -- with one cvt.rn.f16x2.e4m3x2 per pair and
// the query in column 0 only (no per-group scales to keep apart).
template <int H, int D_IDX>
struct Fp8Tile {
    static constexpr int ROW = H * D_IDX;          // bytes per token
    static constexpr int NQL = ROW / 64;           // 64-byte quad loads per token (16 B per lane of a quad)
    static constexpr int QPH = D_IDX / 64;         // quad loads per head
    static_assert(D_IDX % 64 == 0, "d_idx must be a multiple of 64 for the FP8 scoring kernel");
    uint32_t qf[NQL][8];
    float wq[H], ps[H];

    static __device__ __forceinline__ void load_raw(const ScoreArgs& a, int b, int lane, QRaw& r) {
        constexpr int EPL = ROW / 32;
        static_assert(EPL / 8 <= 2, "two 16-byte chunks per lane");
#pragma unroll
        for (int i = 0; i < EPL / 8; ++i)
            r.v[i] = *reinterpret_cast<const uint4*>(a.sel_q + (int64_t)b * ROW + lane * EPL + i * 8);
        r.w = lane < H ? a.w[(int64_t)b * H + lane] : 0.f;
    }
    static __device__ __forceinline__ void stage_raw(const QRaw& r, int lane, uint32_t q16_addr) {
        __half* q16 = reinterpret_cast<__half*>(__cvta_shared_to_generic((size_t)q16_addr));
        float* post = reinterpret_cast<float*>(q16 + ROW);
        constexpr int EPL = ROW / 32, LPH = 32 / H;
        static_assert(EPL % 8 == 0 && LPH * EPL == D_IDX && (LPH & (LPH - 1)) == 0, "query staging geometry");
        __syncwarp();
        float v[EPL], mx = 0.f;
#pragma unroll
        for (int i = 0; i < EPL / 8; ++i) {
            const uint32_t wds[4] = {r.v[i].x, r.v[i].y, r.v[i].z, r.v[i].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) { v[i * 8 + 2 * j] = bf16lo(wds[j]); v[i * 8 + 2 * j + 1] = bf16hi(wds[j]); }
        }
#pragma unroll
        for (int i = 0; i < EPL; ++i) mx = fmaxf(mx, fabsf(v[i]));
#pragma unroll
        for (int o = LPH / 2; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        int sh = 0;
        if (mx > 0.f) sh = 14 - ilogbf(mx);       // E4M3 magnitudes reach 448 = 2^8.8: products stay below 2^24
        sh = max(-100, min(100, sh));
        sh -= 9;                                   // keep |q16| * 448 * d_idx inside fp32-exact accumulation range
        const float up = __uint_as_float((uint32_t)(127 + sh) << 23);
#pragma unroll
        for (int i = 0; i < EPL; ++i) q16[lane * EPL + i] = __float2half_rn(v[i] * up);
        if (lane % LPH == 0) post[lane / LPH] = __uint_as_float((uint32_t)(127 - sh) << 23);
        if (lane < H) post[H + lane] = r.w;
        __syncwarp();
    }
    __device__ __forceinline__ void fetch(int lane, uint32_t q16_addr) {
        const int g = lane >> 2, c = lane & 3;
        const __half* q16 = reinterpret_cast<const __half*>(__cvta_shared_to_generic((size_t)q16_addr));
        const float* post = reinterpret_cast<const float*>(q16 + ROW);
#pragma unroll
        for (int ql = 0; ql < NQL; ++ql)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t* src = reinterpret_cast<const uint32_t*>(q16 + ql * 64 + 16 * c + 4 * j);
                qf[ql][2 * j] = (g == 0) ? src[0] : 0u;
                qf[ql][2 * j + 1] = (g == 0) ? src[1] : 0u;
            }
#pragma unroll
        for (int h = 0; h < H; ++h) { wq[h] = post[H + h]; ps[h] = post[h]; }
    }

    static __device__ __forceinline__ void e4m3x4_to_f16x2x2(uint32_t w, uint32_t& lo, uint32_t& hi) {
        asm("{ .reg .b16 l, h; mov.b32 {l, h}, %2; cvt.rn.f16x2.e4m3x2 %0, l; cvt.rn.f16x2.e4m3x2 %1, h; }"
            : "=r"(lo), "=r"(hi) : "r"(w));
    }

    // maximum over NIT * 16 tokens starting at token t0, whose codes start at shared address st
    // (it0: index of the slice's first 16-token group inside its tile, for the fine form)
    template <int NIT>
    __device__ __forceinline__ float part_max(uint32_t st, int t0, int L, int lane, bool fine, int it0) const {
        const int g = lane >> 2, c = lane & 3;
        float m = -INFINITY;
#pragma unroll 2
        for (int it = 0; it < NIT; ++it) {
            uint4 ca[NQL], cb[NQL];
#pragma unroll
            for (int ql = 0; ql < NQL; ++ql) {
                ca[ql] = lds128(st + (it * 16 + g) * ROW + ql * 64 + c * 16);
                cb[ql] = lds128(st + (it * 16 + 8 + g) * ROW + ql * 64 + c * 16);
            }
            float sa = 0.f, sb = 0.f;
#pragma unroll
            for (int h = 0; h < H; ++h) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int qq = 0; qq < QPH; ++qq) {
                    const int ql = h * QPH + qq;
                    const uint32_t wa[4] = {ca[ql].x, ca[ql].y, ca[ql].z, ca[ql].w};
                    const uint32_t wb[4] = {cb[ql].x, cb[ql].y, cb[ql].z, cb[ql].w};
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        uint32_t a0, a2, a1, a3;
                        e4m3x4_to_f16x2x2(wa[j], a0, a2);
                        e4m3x4_to_f16x2x2(wb[j], a1, a3);
                        mma_f16_16816(acc, a0, a1, a2, a3, qf[ql][2 * j], qf[ql][2 * j + 1]);
                    }
                }
                sa = fmaf(wq[h], fmaxf(acc[0] * ps[h], 0.f), sa);     // column 0, row g     (valid on lanes c == 0)
                sb = fmaf(wq[h], fmaxf(acc[2] * ps[h], 0.f), sb);     // column 0, row g + 8
            }
            const int ta = t0 + it * 16 + g, tb = ta + 8;
            m = group_update(m, sa, sb, ta < L, tb < L, it0 + it, lane, fine);
        }
        return fine ? m : rows_max(m, lane);
    }
};

// block scores of tile t of sequence b: one (lane 0) or, with 16-token blocks, up to four (lanes 0, 4, 8, 12)
__device__ __forceinline__ void store_scores(const ScoreArgs& a, int b, int t, int L, int lane, float m) {
    int j = -1;
    if (a.fine) {
        const int grp = lane >> 2;
        if ((lane & 3) == 0 && grp < 4 && t * 64 + grp * 16 < L) j = t * 4 + grp;
    } else if (lane == 0) {
        j = t;
    }
    if (j >= 0) {
        if (a.tagged) st_tagged_score(a.tagged + (int64_t)b * a.nb_stride + j, a.tag, m);
        else a.scores[(int64_t)b * a.nb_stride + j] = m;
    }
}

template <int H, int D_IDX, int FMT>
__global__ void __launch_bounds__((ScoreCfg<H, D_IDX, FMT>::THREADS), 1) score_decode_kernel(const __grid_constant__ CUtensorMap tm_k,
                                                                     const ScoreArgs a) {
    using Cfg = ScoreCfg<H, D_IDX, FMT>;
    constexpr int NS = Cfg::STAGES;
    constexpr int SC_CONSUMERS = Cfg::CONSUMERS;
    extern __shared__ unsigned char smem_raw[];
    // [0, 256): tile counts of the first 64 sequences (tiles_of); then the ring, 1024-byte aligned
    const uint32_t ring = (smem_u32(smem_raw) + 256u + 1023u) & ~1023u;
    const uint32_t bar_full = ring + NS * Cfg::STAGE_BYTES;        // [NS]
    const uint32_t bar_empty = bar_full + NS * 8;                  // [NS]
    const uint32_t q16_base = bar_empty + NS * 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool fine = a.fine != 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 1); }
        mbar_fence_init();
        if (FMT == SPOT_SELK_BF16) tma_prefetch_desc(&tm_k);
    }
    __syncthreads();
#ifdef SPOT_TRACE
    SPOT_STAMP(a.sync, 0, 0);
#endif
    pdl_wait();
    pdl_launch_dependents();

    // this CTA's work list: its range of every group, in group order
    __shared__ CtaRange s_rng[SC_MAX_GROUPS];
    using TileT = typename std::conditional<FMT == SPOT_SELK_BF16, Bf16Tile<H, D_IDX>,
                  typename std::conditional<FMT == SPOT_SELK_FP8_E4M3, Fp8Tile<H, D_IDX>,
                  typename std::conditional<FMT == SPOT_SELK_MXINT8, Q8Tile<H, D_IDX>, Q4Tile<H, D_IDX, FMT>>::type>::type>::type;
    // the two cold global reads in front of everything -- the sequence lengths and this warp's first query row -- go
    // out together
    const bool q_staged = a.B <= Cfg::Q_SLOTS;
    QRaw raw0;
    const bool have_raw0 = q_staged && warp < SC_CONSUMERS && warp < a.B;
    if (have_raw0) TileT::load_raw(a, warp, lane, raw0);
    if (threadIdx.x < SC_NB_CACHE && (int)threadIdx.x < a.B)
        reinterpret_cast<int*>(smem_raw)[threadIdx.x] = (seq_len_of(a, threadIdx.x) + 63) >> 6;
    __syncthreads();
    if ((int)threadIdx.x < a.n_groups) cta_range_of_group(a, threadIdx.x, s_rng);
    __syncthreads();
    int n_my = 0;
    for (int gg = 0; gg < a.n_groups; ++gg) n_my += s_rng[gg].len;
    if (n_my <= 0) return;
    TileCursor cur;
    cur.first(a, s_rng);
    // queries: staged once per CTA when every sequence has a slot (ScoreCfg), else per warp on every change of sequence.
    // The staging runs AFTER the first tile requests are out (below) and ends on a barrier of the consumer warps only.
    auto stage_queries = [&]() {
        if (!q_staged) return;
        for (int bb = warp; bb < a.B; bb += SC_CONSUMERS) {
            if (bb != warp) TileT::load_raw(a, bb, lane, raw0);
            TileT::stage_raw(raw0, lane, q16_base + bb * Cfg::Q_SLOT_BYTES);
        }
        asm volatile("bar.sync 1, %0;" :: "n"(SC_CONSUMERS * 32) : "memory");
    };
    auto take_query = [&](TileT& tile, int bb) {
        if (q_staged) { tile.fetch(lane, q16_base + bb * Cfg::Q_SLOT_BYTES); return; }
        __syncwarp();
        QRaw r;
        TileT::load_raw(a, bb, lane, r);
        TileT::stage_raw(r, lane, q16_base + warp * Cfg::Q_SLOT_BYTES);
        tile.fetch(lane, q16_base + warp * Cfg::Q_SLOT_BYTES);
        __syncwarp();
    };

    if constexpr (Cfg::SELF) {
        // ================================ self-serve consumers (4-bit) ================================
        // warp w streams tiles w, w + C, w + 2C, ... through its own stages w*K .. w*K + K-1
        // (a stage holds one of the SP slices of a tile; SP == 1 for the 4-bit formats)
        constexpr int K = Cfg::PER_WARP, SP = Cfg::SPLIT;
        TileT tile;
        cur.advance(a, s_rng, warp);
        TileCursor nxt = cur;                      // the tile of the next slice to request
        const int n_w = (n_my - warp + SC_CONSUMERS - 1) / SC_CONSUMERS;     // tiles of this warp
        const int n_q = n_w * SP;                  // slices of this warp
        int rq = 0;                                // next slice to request: slice q -> stage w*K + q % K
        auto request_next = [&]() {
            if (rq >= n_q) return;
            if (lane == 0) {
                const uint32_t s = warp * K + rq % K;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic reads of the stage
                mbar_arrive_expect_tx(bar_full + 8 * s, Cfg::STAGE_BYTES);
                const uint8_t* tile_src = a.sel_k + ((int64_t)nxt.b * a.tiles_per_seq + nxt.t) * Cfg::TILE_BYTES;
                if constexpr (FMT == SPOT_SELK_FP8_E4M3 || SP == 1) {
                    bulk_load(ring + s * Cfg::STAGE_BYTES, tile_src + (rq % SP) * Cfg::STAGE_BYTES, Cfg::STAGE_BYTES,
                              bar_full + 8 * s);
                } else {
                    // 4-bit slice: the slice's code rows, then its scale rows (they sit behind all 64 code rows)
                    constexpr int NTOK = 64 / SP, CODES = NTOK * Cfg::CODE_BYTES, SCALES = NTOK * Cfg::SCALE_BYTES;
                    static_assert(CODES + SCALES == Cfg::STAGE_BYTES && SCALES % 16 == 0, "4-bit slice geometry");
                    bulk_load(ring + s * Cfg::STAGE_BYTES, tile_src + (rq % SP) * CODES, CODES, bar_full + 8 * s);
                    bulk_load(ring + s * Cfg::STAGE_BYTES + CODES, tile_src + SP * CODES + (rq % SP) * SCALES, SCALES,
                              bar_full + 8 * s);
                }
            }
            if (rq % SP == SP - 1) nxt.advance(a, s_rng, SC_CONSUMERS);
            ++rq;
        };
#ifdef SPOT_TRACE
        if (warp == 0) SPOT_STAMP(a.sync, 6, 0);
#endif
#pragma unroll
        for (int j = 0; j < K; ++j) request_next();
        stage_queries();
#ifdef SPOT_TRACE
        if (warp == 0) SPOT_STAMP(a.sync, 6, 1);
#endif
        int cur_b = -1, L = 0;
        for (int j = 0; j < n_w; ++j) {
            if (cur.b != cur_b) {
                cur_b = cur.b;
                L = seq_len_of(a, cur_b);
                take_query(tile, cur_b);
            }
            float m = -INFINITY;
#pragma unroll
            for (int part = 0; part < SP; ++part) {
                const int q = j * SP + part;
                const uint32_t s = warp * K + q % K;
                mbar_wait(bar_full + 8 * s, (q / K) & 1);
#ifdef SPOT_TRACE
                if (warp == 0 && q == 0) SPOT_STAMP(a.sync, 6, 2);
                if (warp == 0 && q == 2) SPOT_STAMP(a.sync, 6, 3);
#endif
                m = fmaxf(m, tile.template part_max<4 / SP>(ring + s * Cfg::STAGE_BYTES, cur.t * 64 + part * (64 / SP),
                                                            L, lane, fine, part * (4 / SP)));
                __syncwarp();
                request_next();
            }
            store_scores(a, cur_b, cur.t, L, lane, m);
            cur.advance(a, s_rng, SC_CONSUMERS);
        }
    } else if (warp == SC_CONSUMERS) {
        // ================================ producer ================================
        if (lane == 0) {
            for (int i = 0; i < n_my; ++i) {
                const int s = i % NS;
                mbar_wait(bar_empty + 8 * s, ((i / NS) & 1) ^ 1);
                mbar_arrive_expect_tx(bar_full + 8 * s, Cfg::TILE_BYTES);
                if (FMT == SPOT_SELK_BF16)
                    tma_load_4d(ring + s * Cfg::STAGE_BYTES, &tm_k, bar_full + 8 * s, 0, cur.t * 64, 0, cur.b);
                else
                    bulk_load(ring + s * Cfg::STAGE_BYTES,
                              a.sel_k + ((int64_t)cur.b * a.tiles_per_seq + cur.t) * Cfg::TILE_BYTES, Cfg::TILE_BYTES,
                              bar_full + 8 * s);
                cur.advance(a, s_rng, 1);
            }
        }
    } else {
        // ================================ consumers ================================
        TileT tile;
        cur.advance(a, s_rng, warp);
        stage_queries();
        int cur_b = -1, L = 0;
        for (int i = warp; i < n_my; i += SC_CONSUMERS) {
            if (cur.b != cur_b) {
                cur_b = cur.b;
                L = seq_len_of(a, cur_b);
                take_query(tile, cur_b);
            }
            const int s = i % NS;
#ifdef SPOT_TRACE
            if (warp == 0 && i == 0) SPOT_STAMP(a.sync, 6, 0);
#endif
            mbar_wait(bar_full + 8 * s, (i / NS) & 1);
#ifdef SPOT_TRACE
            if (warp == 0 && i < 3 * SC_CONSUMERS) SPOT_STAMP(a.sync, 6, 1 + i / SC_CONSUMERS);
#endif
            const float m = tile.tile_max(ring + s * Cfg::STAGE_BYTES, cur.t * 64, L, lane, fine);
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * s);
            store_scores(a, cur_b, cur.t, L, lane, m);
            cur.advance(a, s_rng, SC_CONSUMERS);
        }
    }
#ifdef SPOT_TRACE
    __syncthreads();
    SPOT_STAMP(a.sync, 0, 2);
#endif
}

// sync: hand-offs of a pipelined step (nullptr: none) -- `scores` is then the [B][nb_stride] array of tagged 64-bit words.
// reserve_sms: SMs left to the selection CTAs that run beside this kernel.
template <int H, int D_IDX, int FMT>
spot_status launch_score_fmt(const spot_select_params* p, float* scores, int nb_stride, const StepSync* sync, int reserve_sms,
                             cudaStream_t s) {
    using Cfg = ScoreCfg<H, D_IDX, FMT>;
    ScoreArgs a;
    a.sel_q = p->sel_q; a.w = p->w; a.sel_k = (const uint8_t*)p->sel_k; a.tiles_per_seq = p->cache_stride_tokens / 64;
    a.seq_len = p->seq_len; a.max_len = p->max_seq_len; a.B = p->B; a.n_groups = p->B < 4 ? p->B : 4; a.scores = scores; a.nb_stride = nb_stride; a.fine = p->blk == 16;
    CUtensorMap tm;
    memset(&tm, 0, sizeof(tm));
    if (FMT == SPOT_SELK_BF16) {
        constexpr int NP = H * D_IDX / 64;
        const uint64_t row_bytes = (uint64_t)H * D_IDX * 2;
        const uint64_t dims[4] = {64, (uint64_t)p->cache_stride_tokens, (uint64_t)NP, (uint64_t)p->B};
        const uint64_t strides[3] = {row_bytes, 128, (uint64_t)p->cache_stride_tokens * row_bytes};
        const uint32_t box[4] = {64, 64, (uint32_t)NP, 1};
        if (!encode_tmap_bf16_sw128(&tm, p->sel_k, 4, dims, strides, box)) return SPOT_ERR_CUDA;
    }
    static unsigned long long smem_attr_done = 0;
    SPOT_CUDA_TRY(set_max_smem_once(score_decode_kernel<H, D_IDX, FMT>, Cfg::SMEM_BYTES, smem_attr_done));
    const int64_t max_tiles = (int64_t)p->B * ((p->max_seq_len + 63) / 64);
    const int sms = sm_count() - reserve_sms > 0 ? sm_count() - reserve_sms : 1;
    const int grid = (int)(max_tiles < sms ? max_tiles : sms);
    a.tagged = nullptr; a.tag = 0;
    if (sync && sync->tag) { a.tagged = reinterpret_cast<unsigned long long*>(scores); a.tag = sync->tag; a.scores = nullptr; }
#ifdef SPOT_TRACE
    memset(&a.sync, 0, sizeof(a.sync));
    if (sync) a.sync = *sync;
#endif
    SPOT_CUDA_TRY(launch_pdl(score_decode_kernel<H, D_IDX, FMT>, dim3((unsigned)grid), dim3(Cfg::THREADS),
                             (size_t)Cfg::SMEM_BYTES, s, tm, a));
    return SPOT_OK;
}

template <int H, int D_IDX>
spot_status launch_score(const spot_select_params* p, float* scores, int nb_stride, const StepSync* sync, int reserve_sms,
                         cudaStream_t s) {
    if (p->fmt == SPOT_SELK_BF16) return launch_score_fmt<H, D_IDX, SPOT_SELK_BF16>(p, scores, nb_stride, sync, reserve_sms, s);
    if (p->fmt == SPOT_SELK_MXFP4) return launch_score_fmt<H, D_IDX, SPOT_SELK_MXFP4>(p, scores, nb_stride, sync, reserve_sms, s);
    if (p->fmt == SPOT_SELK_FP8_E4M3)
        return launch_score_fmt<H, D_IDX, SPOT_SELK_FP8_E4M3>(p, scores, nb_stride, sync, reserve_sms, s);
    if (p->fmt == SPOT_SELK_MXINT8) return launch_score_fmt<H, D_IDX, SPOT_SELK_MXINT8>(p, scores, nb_stride, sync, reserve_sms, s);
    if (p->fmt == SPOT_SELK_INT4_BF16S)
        return launch_score_fmt<H, D_IDX, SPOT_SELK_INT4_BF16S>(p, scores, nb_stride, sync, reserve_sms, s);
    return launch_score_fmt<H, D_IDX, SPOT_SELK_INT4_E4M3>(p, scores, nb_stride, sync, reserve_sms, s);
}

}  // namespace

// scores: fp32 [B][nb_stride]
spot_status score_decode(const spot_select_params* p, float* scores, int nb_stride, const StepSync* sync, int reserve_sms,
                         cudaStream_t s) {
    if (p->H_idx == 4 && p->d_idx == 64) return launch_score<4, 64>(p, scores, nb_stride, sync, reserve_sms, s);
    if (p->H_idx == 4 && p->d_idx == 128) return launch_score<4, 128>(p, scores, nb_stride, sync, reserve_sms, s);
    return SPOT_ERR_UNSUPPORTED;
}

}  // namespace spot
