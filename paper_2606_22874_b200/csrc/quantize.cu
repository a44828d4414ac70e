// Step a0 -- group-32 "microscale" quantisers of the selector K-cache (
// definitions: DESIGN.md R16).  One thread per 32-element group: 64 B in (4 x LDG.128), 16 B + 1 B out.
// HBM-bound streaming pass (512 B read + 136 B written per token at H_idx x d_idx = 4 x 64).
//
// Opaque tile layout (SELK_TILE = 64 tokens per tile):
//   tile = [64][H*d/2] code bytes | [64][H*d/32] scale bytes
//   MXFP4 : byte P of a group = E2M1(dim 2P) | E2M1(dim 2P+1) << 4           (what cvt.e2m1x2 unpacks)
//   INT4  : offset-binary u = q + 8; 32-bit word wd of a group holds dims 8wd..8wd+7 with
//           dim 8wd + 2pp + e at nibble pp + 4e, so that (w >> 4pp) & 0x000F000F is the pair (2pp, 2pp+1)
//           (what the fp16 magic-number unpack in score_decode.cu wants).
//   INT4_BF16S (f2, R39): INT4's codes; the scale rows hold two bytes per group (the BF16 bits of the scale).
//   MXINT8 (f2, R38): [64][H*d] code bytes | [64][H*d/32] E8M0 bytes.  A code byte is offset-binary u = code + 128
//           (read as an fp16 subnormal by the scoring kernel, the offset taken on the query side).  Every 128 bytes of a
//           token's codes are four groups as two 64-byte halves -- half hh holds bytes [16 hh, 16 hh + 16) of each of the
//           four groups -- and ODD tokens store the two halves swapped, so that the 16-byte shared-memory loads of two
//           adjacent token rows fall into different banks.
#include <cuda_bf16.h>
#include <cuda_fp8.h>

#include "common.cuh"

namespace spot {

namespace {

__device__ __forceinline__ uint32_t e2m1x2_from_f32(float lo, float hi) {
    // cvt.rn.satfinite.e2m1x2.f32 d, a, b : a -> upper nibble, b -> lower nibble.  RNE on the E2M1 grid,
    // saturating at +-6, keeps the sign of a zero result (R16; checked bit-for-bit against the
    // oracle's threshold table in tests/test_gpu_decode.py::test_quantise_dequantise_bit_exact, ties included).
    uint32_t r;
    asm("{ .reg .b8 t; cvt.rn.satfinite.e2m1x2.f32 t, %1, %2; cvt.u32.u8 %0, t; }" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

__device__ __forceinline__ float e4m3_to_f32(uint32_t code) {
    __half_raw h = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)code, __NV_E4M3);
    return __half2float(*reinterpret_cast<__half*>(&h));
}

template <int FMT>
__global__ void __launch_bounds__(256) quantize_kernel(const uint16_t* __restrict__ k_in, uint8_t* __restrict__ cache,
                                                       int64_t n_tokens, int64_t token_offset, int64_t tiles_per_seq,
                                                       int groups_per_token, int64_t total_groups,
                                                       const int32_t* __restrict__ pos) {
    pdl_wait();
    int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total_groups) return;
    int gi = (int)(gid % groups_per_token);
    int64_t tok_lin = gid / groups_per_token;            // b * n_tokens + t
    int64_t b = tok_lin / n_tokens;
    int64_t t = token_offset + (tok_lin - b * n_tokens);
    if (pos) {                                           // append form: one token per sequence at its own slot
        t = pos[b];
        if (t < 0 || t >= tiles_per_seq * SELK_TILE) return;
    }

    const uint4* src = reinterpret_cast<const uint4*>(k_in + gid * 32);
    uint32_t wv[16];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint4 x = ldg_stream_v4(src + i);
        wv[4 * i + 0] = x.x; wv[4 * i + 1] = x.y; wv[4 * i + 2] = x.z; wv[4 * i + 3] = x.w;
    }
    float v[32];
    float amax = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        v[2 * i] = bf16lo(wv[i]);
        v[2 * i + 1] = bf16hi(wv[i]);
        amax = fmaxf(amax, fmaxf(fabsf(v[2 * i]), fabsf(v[2 * i + 1])));
    }

    constexpr int CB = selk_code_bytes_per_group(FMT), SB = selk_scale_bytes_per_group(FMT);
    uint32_t out[CB / 4];
    uint32_t scale_bits;
    if (FMT == SPOT_SELK_MXFP4) {
        // e = floor(log2 amax) - 2 clamped to [-127, 127]; X = 2^e; code = RNE_E2M1(v / X), saturating.
        int e = 0;
        if (amax > 0.f) {
            e = ilogbf(amax) - 2;
            e = max(-127, min(127, e));
        }
        scale_bits = (uint32_t)(e + 127);
        // 1/X = 2^-e, -e in [-125(+2), 127]: always a normal binary32 except e = 127 (unreachable: e <= 125).
        float inv = __uint_as_float((uint32_t)(127 - e) << 23);
        if (e == 127) inv = __uint_as_float(0x00400000u);   // 2^-127 (kept for completeness)
#pragma unroll
        for (int wd = 0; wd < 4; ++wd) {
            uint32_t acc = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                int P = wd * 4 + j;
                acc |= e2m1x2_from_f32(v[2 * P] * inv, v[2 * P + 1] * inv) << (8 * j);
            }
            out[wd] = acc;
        }
    } else if (FMT == SPOT_SELK_MXINT8) {
        // e = floor(log2 amax) clamped to [-127, 127]; code = clamp(RNE(v 2^(6 - e)), -127, 127); stored as u = code + 128.
        int e = 0;
        if (amax > 0.f) e = max(-127, min(127, ilogbf(amax)));
        scale_bits = (uint32_t)(e + 127);
#pragma unroll
        for (int wd = 0; wd < 8; ++wd) {
            uint32_t acc = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float r = fminf(fmaxf(rintf(scalbnf(v[4 * wd + j], 6 - e)), -127.f), 127.f);   // scalbnf: exact
                acc |= (uint32_t)((int)r + 128) << (8 * j);
            }
            out[wd] = acc;
        }
    } else {
        // sf = amax / 7 (binary32 RNE); INT4_E4M3: code = E4M3_rne_satfinite(sf); INT4_BF16S: the BF16 nearest sf; either
        // bumped to its smallest subnormal if it rounds to 0 with amax > 0; q = clamp(rint(v / s), -7, 7) with
        // s = value(scale); stored as u = q + 8.
        float sf = __fdiv_rn(amax, 7.0f);
        float s;
        if (FMT == SPOT_SELK_INT4_BF16S) {
            uint32_t sb = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(sf));
            if (sb == 0 && amax > 0.f) sb = 1;
            scale_bits = sb;
            s = __uint_as_float(sb << 16);
        } else {
            uint32_t code = (uint32_t)__nv_cvt_float_to_fp8(sf, __NV_SATFINITE, __NV_E4M3) & 0xffu;
            if (code == 0 && amax > 0.f) code = 1;
            scale_bits = code;
            s = e4m3_to_f32(code);
        }
#pragma unroll
        for (int wd = 0; wd < 4; ++wd) {
            uint32_t acc = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float x = v[8 * wd + j];
                float tq = (s > 0.f) ? __fdiv_rn(x, s) : 0.f;
                float r = fminf(fmaxf(rintf(tq), -7.f), 7.f);
                uint32_t u = (uint32_t)((int)r + 8);
                int pp = j >> 1, e = j & 1;
                acc |= u << (4 * (pp + 4 * e));
            }
            out[wd] = acc;
        }
    }

    int64_t tile = t / SELK_TILE;
    int r = (int)(t % SELK_TILE);
    int64_t cpt = (int64_t)groups_per_token * CB;
    int64_t spt = (int64_t)groups_per_token * SB;
    uint8_t* tile_base = cache + (b * tiles_per_seq + tile) * (SELK_TILE * (cpt + spt));
    if (FMT == SPOT_SELK_MXINT8) {
        uint8_t* unit = tile_base + r * cpt + (gi >> 2) * 128 + (gi & 3) * 16;
        *reinterpret_cast<uint4*>(unit + ((r & 1) ? 64 : 0)) = make_uint4(out[0], out[1], out[2], out[3]);
        *reinterpret_cast<uint4*>(unit + ((r & 1) ? 0 : 64)) = make_uint4(out[CB / 4 - 4], out[CB / 4 - 3], out[CB / 4 - 2], out[CB / 4 - 1]);
    } else {
        *reinterpret_cast<uint4*>(tile_base + r * cpt + gi * 16) = make_uint4(out[0], out[1], out[2], out[3]);
    }
    if (SB == 2) *reinterpret_cast<uint16_t*>(tile_base + SELK_TILE * cpt + r * spt + gi * 2) = (uint16_t)scale_bits;
    else tile_base[SELK_TILE * cpt + r * spt + gi] = (uint8_t)scale_bits;
}

template <int FMT>
__global__ void __launch_bounds__(256) dequantize_kernel(const uint8_t* __restrict__ cache, uint16_t* __restrict__ k_out,
                                                         int64_t n_tokens, int64_t token_offset, int64_t tiles_per_seq,
                                                         int groups_per_token, int64_t total_groups) {
    int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total_groups) return;
    int gi = (int)(gid % groups_per_token);
    int64_t tok_lin = gid / groups_per_token;
    int64_t b = tok_lin / n_tokens;
    int64_t t = token_offset + (tok_lin - b * n_tokens);
    int64_t tile = t / SELK_TILE;
    int r = (int)(t % SELK_TILE);
    constexpr int CB = selk_code_bytes_per_group(FMT), SB = selk_scale_bytes_per_group(FMT);
    int64_t cpt = (int64_t)groups_per_token * CB;
    int64_t spt = (int64_t)groups_per_token * SB;
    const uint8_t* tile_base = cache + (b * tiles_per_seq + tile) * (SELK_TILE * (cpt + spt));
    uint32_t w[CB / 4];
    if (FMT == SPOT_SELK_MXINT8) {
        const uint8_t* unit = tile_base + r * cpt + (gi >> 2) * 128 + (gi & 3) * 16;
        const uint4 lo = *reinterpret_cast<const uint4*>(unit + ((r & 1) ? 64 : 0));
        const uint4 hi = *reinterpret_cast<const uint4*>(unit + ((r & 1) ? 0 : 64));
        w[0] = lo.x; w[1] = lo.y; w[2] = lo.z; w[3] = lo.w;
        w[CB / 4 - 4] = hi.x; w[CB / 4 - 3] = hi.y; w[CB / 4 - 2] = hi.z; w[CB / 4 - 1] = hi.w;
    } else {
        const uint4 c = *reinterpret_cast<const uint4*>(tile_base + r * cpt + gi * 16);
        w[0] = c.x; w[1] = c.y; w[2] = c.z; w[3] = c.w;
    }
    const uint32_t sb = SB == 2 ? (uint32_t)*reinterpret_cast<const uint16_t*>(tile_base + SELK_TILE * cpt + r * spt + gi * 2)
                                : (uint32_t)tile_base[SELK_TILE * cpt + r * spt + gi];
    float v[32];
    if (FMT == SPOT_SELK_MXFP4) {
        float X = sb ? __uint_as_float(sb << 23) : __uint_as_float(0x00400000u);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            uint32_t code = (w[i >> 3] >> (4 * (i & 7))) & 0xf;
            uint32_t m = code & 7;
            // E2M1 magnitudes: s e e m -> e == 0 ? 0.5 m : 2^(e-1) (1 + m/2)
            uint32_t e = m >> 1, mm = m & 1;
            float mag = e == 0 ? 0.5f * (float)mm : (float)(1u << (e - 1)) * (1.f + 0.5f * (float)mm);
            float val = mag * X;
            v[i] = (code & 8) ? -val : val;
        }
    } else if (FMT == SPOT_SELK_MXINT8) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const int code = (int)((w[i >> 2] >> (8 * (i & 3))) & 0xffu) - 128;
            v[i] = scalbnf((float)code, (int)sb - 127 - 6) + 0.0f;          // exact: <= 7 significant bits
        }
    } else {
        float s = FMT == SPOT_SELK_INT4_BF16S ? __uint_as_float(sb << 16) : e4m3_to_f32(sb);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            int wd = i >> 3, j = i & 7, pp = j >> 1, e = j & 1;
            int q = (int)((w[wd] >> (4 * (pp + 4 * e))) & 0xf) - 8;
            v[i] = (float)q * s + 0.0f;                                    // exact in fp32 (3 x 8 significant bits)
        }
    }
    uint32_t o[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        if (FMT == SPOT_SELK_INT4_BF16S) {
            // up to 11 significant bits: the BF16 view is a rounding (R39; a diagnostic -- the scoring kernel uses q * s)
            o[i] = pack_bf16x2(v[2 * i], v[2 * i + 1]);
        } else {
            // exact: every dequantised value has <= 8 significant bits (R16), so truncation == the value
            o[i] = (__float_as_uint(v[2 * i]) >> 16) | (__float_as_uint(v[2 * i + 1]) & 0xffff0000u);
        }
    }
    uint4* dst = reinterpret_cast<uint4*>(k_out + gid * 32);
#pragma unroll
    for (int i = 0; i < 4; ++i) dst[i] = make_uint4(o[4 * i], o[4 * i + 1], o[4 * i + 2], o[4 * i + 3]);
}

// f2 -- FP8-E4M3 per element (R30): cache [B][tokens][H*d] bytes, byte = cvt.rn.satfinite.e4m3x2.f32 of
// the element (RNE onto the E4M3 grid, saturating at +-448, sign of zero kept); 16 elements per thread.
__global__ void __launch_bounds__(256) fp8_quantize_kernel(const uint16_t* __restrict__ k_in, uint8_t* __restrict__ cache,
                                                           int64_t n_tokens, int64_t token_offset, int64_t stride_tokens,
                                                           int64_t vec_per_token, int64_t total,
                                                           const int32_t* __restrict__ pos) {
    pdl_wait();
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int64_t per_seq = n_tokens * vec_per_token;
    const int64_t b = i / per_seq, r = i - b * per_seq;
    int64_t t = token_offset + r / vec_per_token;
    if (pos) {
        t = pos[b];
        if (t < 0 || t >= stride_tokens) return;
    }
    const uint4* src = reinterpret_cast<const uint4*>(k_in + i * 16);
    const uint4 x0 = ldg_stream_v4(src), x1 = ldg_stream_v4(src + 1);
    const uint32_t w[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
    uint32_t o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(bf16lo(w[2 * j]), bf16hi(w[2 * j])), __NV_SATFINITE, __NV_E4M3);
        const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(bf16lo(w[2 * j + 1]), bf16hi(w[2 * j + 1])), __NV_SATFINITE, __NV_E4M3);
        o[j] = (lo & 0xffffu) | (hi << 16);
    }
    *reinterpret_cast<uint4*>(cache + ((b * stride_tokens + t) * vec_per_token + r % vec_per_token) * 16) =
        make_uint4(o[0], o[1], o[2], o[3]);
}

__global__ void __launch_bounds__(256) fp8_dequantize_kernel(const uint8_t* __restrict__ cache, uint16_t* __restrict__ k_out,
                                                             int64_t n_tokens, int64_t token_offset, int64_t stride_tokens,
                                                             int64_t vec_per_token, int64_t total) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int64_t per_seq = n_tokens * vec_per_token;
    const int64_t b = i / per_seq, r = i - b * per_seq;
    const int64_t t = token_offset + r / vec_per_token;
    const uint4 c = *reinterpret_cast<const uint4*>(cache + ((b * stride_tokens + t) * vec_per_token + r % vec_per_token) * 16);
    const uint32_t cw[4] = {c.x, c.y, c.z, c.w};
    uint32_t o[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)((cw[j >> 1] >> (16 * (j & 1))) & 0xffffu), __NV_E4M3);
        const float lo = __half2float(__ushort_as_half(h.x)), hi = __half2float(__ushort_as_half(h.y));
        o[j] = pack_bf16x2(lo, hi);                       // exact: E4M3 values have 4 significant bits
    }
    uint4* dst = reinterpret_cast<uint4*>(k_out + i * 16);
    dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
    dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
}

// BF16 "format": plain row copy into / out of the cache (16 B per thread).
__global__ void __launch_bounds__(256) copy_rows_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst,
                                                        int64_t n_tokens, int64_t vec_per_token,
                                                        int64_t src_stride_tokens, int64_t src_offset,
                                                        int64_t dst_stride_tokens, int64_t dst_offset, int64_t total,
                                                        const int32_t* __restrict__ pos) {
    pdl_wait();
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    int64_t per_seq = n_tokens * vec_per_token;
    int64_t b = i / per_seq, r = i - b * per_seq;
    if (pos) {
        dst_offset = pos[b];
        if (dst_offset < 0 || dst_offset >= dst_stride_tokens) return;
    }
    dst[(b * dst_stride_tokens + dst_offset) * vec_per_token + r] =
        src[(b * src_stride_tokens + src_offset) * vec_per_token + r];
}

spot_status check_quant_args(const void* a, const void* b, int fmt, int64_t B, int64_t n_tokens, int64_t token_offset,
                             int64_t stride, int H, int d) {
    if (!a || !b || !aligned16(a) || !aligned16(b)) return SPOT_ERR_INVALID_ARG;
    if (!selk_is_format(fmt)) return SPOT_ERR_INVALID_ARG;
    if (B <= 0 || n_tokens <= 0 || token_offset < 0 || H <= 0 || d <= 0 || d % 32 != 0) return SPOT_ERR_INVALID_ARG;
    if (token_offset + n_tokens > stride) return SPOT_ERR_INVALID_ARG;
    if (fmt != SPOT_SELK_BF16 && stride % SELK_TILE != 0) return SPOT_ERR_INVALID_ARG;
    return SPOT_OK;
}

}  // namespace

// f1: write one new token per sequence (k_new [B][H*d] BF16) into the cache at slot pos[b] (device array), in format fmt.
// Same quantisers, same layout; launched with the PDL attribute so that it chains behind the projection kernel.
spot_status append_selector_k(const uint16_t* k_new, void* cache, int fmt, int B, const int32_t* pos, int64_t stride,
                              int H, int d, cudaStream_t s) {
    if (fmt == SPOT_SELK_BF16) {
        const int64_t vpt = (int64_t)H * d / 8, total = (int64_t)B * vpt;
        SPOT_CUDA_TRY(launch_pdl(copy_rows_kernel, dim3((unsigned)ceil_div64(total, 256)), dim3(256), 0, s,
                                 (const uint4*)k_new, (uint4*)cache, (int64_t)1, vpt, (int64_t)1, (int64_t)0, stride,
                                 (int64_t)0, total, pos));
        return SPOT_OK;
    }
    if (fmt == SPOT_SELK_FP8_E4M3) {
        const int64_t vpt = (int64_t)H * d / 16, total = (int64_t)B * vpt;
        SPOT_CUDA_TRY(launch_pdl(fp8_quantize_kernel, dim3((unsigned)ceil_div64(total, 256)), dim3(256), 0, s, k_new,
                                 (uint8_t*)cache, (int64_t)1, (int64_t)0, stride, vpt, total, pos));
        return SPOT_OK;
    }
    const int gpt = H * d / 32;
    const int64_t total = (int64_t)B * gpt, tiles = stride / SELK_TILE;
    const dim3 grid((unsigned)ceil_div64(total, 256));
#define SPOT_APPEND_AS(F)                                                                                              \
    SPOT_CUDA_TRY(launch_pdl(quantize_kernel<F>, grid, dim3(256), 0, s, k_new, (uint8_t*)cache, (int64_t)1, (int64_t)0, tiles, \
                             gpt, total, pos))
    if (fmt == SPOT_SELK_MXFP4) SPOT_APPEND_AS(SPOT_SELK_MXFP4);
    else if (fmt == SPOT_SELK_MXINT8) SPOT_APPEND_AS(SPOT_SELK_MXINT8);
    else if (fmt == SPOT_SELK_INT4_BF16S) SPOT_APPEND_AS(SPOT_SELK_INT4_BF16S);
    else SPOT_APPEND_AS(SPOT_SELK_INT4_E4M3);
#undef SPOT_APPEND_AS
    return SPOT_OK;
}

}  // namespace spot

using namespace spot;

extern "C" size_t spot_selector_k_bytes(spot_selk_format fmt, int64_t B, int64_t tokens, int H_idx, int d_idx) {
    if (B <= 0 || tokens <= 0 || H_idx <= 0 || d_idx <= 0 || d_idx % 32 != 0) return 0;
    int64_t n = B * tokens * H_idx * d_idx;
    if (fmt == SPOT_SELK_BF16) return (size_t)(2 * n);
    if (selk_is_grouped(fmt)) {
        if (tokens % SELK_TILE != 0) return 0;
        return (size_t)(n / 32 * (selk_code_bytes_per_group(fmt) + selk_scale_bytes_per_group(fmt)));
    }
    if (fmt == SPOT_SELK_FP8_E4M3) return tokens % SELK_TILE != 0 ? 0 : (size_t)n;
    return 0;
}

extern "C" spot_status spot_quantize_selector_k(const uint16_t* k_bf16, void* k_cache, spot_selk_format fmt, int64_t B,
                                                int64_t n_tokens, int64_t token_offset, int64_t cache_stride_tokens,
                                                int H_idx, int d_idx, void* stream) {
    spot_status st = check_quant_args(k_bf16, k_cache, fmt, B, n_tokens, token_offset, cache_stride_tokens, H_idx, d_idx);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    if (fmt == SPOT_SELK_BF16) {
        int64_t vpt = (int64_t)H_idx * d_idx / 8, total = B * n_tokens * vpt;
        copy_rows_kernel<<<(unsigned)ceil_div64(total, 256), 256, 0, s>>>(
            (const uint4*)k_bf16, (uint4*)k_cache, n_tokens, vpt, n_tokens, 0, cache_stride_tokens, token_offset, total, nullptr);
        SPOT_LAUNCH_CHECK();
        return SPOT_OK;
    }
    if (fmt == SPOT_SELK_FP8_E4M3) {
        const int64_t vpt = (int64_t)H_idx * d_idx / 16, total = B * n_tokens * vpt;
        fp8_quantize_kernel<<<(unsigned)ceil_div64(total, 256), 256, 0, s>>>(k_bf16, (uint8_t*)k_cache, n_tokens, token_offset,
                                                                             cache_stride_tokens, vpt, total, nullptr);
        SPOT_LAUNCH_CHECK();
        return SPOT_OK;
    }
    int gpt = H_idx * d_idx / 32;
    int64_t total = B * n_tokens * gpt;
    int64_t tiles = cache_stride_tokens / SELK_TILE;
    unsigned grid = (unsigned)ceil_div64(total, 256);
#define SPOT_QUANT_AS(F) quantize_kernel<F><<<grid, 256, 0, s>>>(k_bf16, (uint8_t*)k_cache, n_tokens, token_offset, tiles, gpt, total, nullptr)
    if (fmt == SPOT_SELK_MXFP4) SPOT_QUANT_AS(SPOT_SELK_MXFP4);
    else if (fmt == SPOT_SELK_MXINT8) SPOT_QUANT_AS(SPOT_SELK_MXINT8);
    else if (fmt == SPOT_SELK_INT4_BF16S) SPOT_QUANT_AS(SPOT_SELK_INT4_BF16S);
    else SPOT_QUANT_AS(SPOT_SELK_INT4_E4M3);
#undef SPOT_QUANT_AS
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}

extern "C" spot_status spot_dequantize_selector_k(const void* k_cache, uint16_t* k_bf16_out, spot_selk_format fmt,
                                                  int64_t B, int64_t n_tokens, int64_t token_offset,
                                                  int64_t cache_stride_tokens, int H_idx, int d_idx, void* stream) {
    spot_status st = check_quant_args(k_cache, k_bf16_out, fmt, B, n_tokens, token_offset, cache_stride_tokens, H_idx, d_idx);
    if (st != SPOT_OK) return st;
    if ((st = check_device()) != SPOT_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    if (fmt == SPOT_SELK_BF16) {
        int64_t vpt = (int64_t)H_idx * d_idx / 8, total = B * n_tokens * vpt;
        copy_rows_kernel<<<(unsigned)ceil_div64(total, 256), 256, 0, s>>>(
            (const uint4*)k_cache, (uint4*)k_bf16_out, n_tokens, vpt, cache_stride_tokens, token_offset, n_tokens, 0, total, nullptr);
        SPOT_LAUNCH_CHECK();
        return SPOT_OK;
    }
    if (fmt == SPOT_SELK_FP8_E4M3) {
        const int64_t vpt = (int64_t)H_idx * d_idx / 16, total = B * n_tokens * vpt;
        fp8_dequantize_kernel<<<(unsigned)ceil_div64(total, 256), 256, 0, s>>>((const uint8_t*)k_cache, k_bf16_out, n_tokens,
                                                                               token_offset, cache_stride_tokens, vpt, total);
        SPOT_LAUNCH_CHECK();
        return SPOT_OK;
    }
    int gpt = H_idx * d_idx / 32;
    int64_t total = B * n_tokens * gpt;
    int64_t tiles = cache_stride_tokens / SELK_TILE;
    unsigned grid = (unsigned)ceil_div64(total, 256);
#define SPOT_DEQUANT_AS(F) dequantize_kernel<F><<<grid, 256, 0, s>>>((const uint8_t*)k_cache, k_bf16_out, n_tokens, token_offset, tiles, gpt, total)
    if (fmt == SPOT_SELK_MXFP4) SPOT_DEQUANT_AS(SPOT_SELK_MXFP4);
    else if (fmt == SPOT_SELK_MXINT8) SPOT_DEQUANT_AS(SPOT_SELK_MXINT8);
    else if (fmt == SPOT_SELK_INT4_BF16S) SPOT_DEQUANT_AS(SPOT_SELK_INT4_BF16S);
    else SPOT_DEQUANT_AS(SPOT_SELK_INT4_E4M3);
#undef SPOT_DEQUANT_AS
    SPOT_LAUNCH_CHECK();
    return SPOT_OK;
}
