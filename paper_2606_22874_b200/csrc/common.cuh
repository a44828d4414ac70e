// Shared device/host helpers of the SpotAttention sm_100a library (product side only; the oracle
// shares nothing with this file).
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/spot.h"

namespace spot {

// ---- host-side status plumbing -------------------------------------------------------------------
void set_last_cuda_error(int e);

#define SPOT_CUDA_TRY(expr)                                  \
    do {                                                     \
        cudaError_t _e = (expr);                             \
        if (_e != cudaSuccess) {                             \
            ::spot::set_last_cuda_error((int)_e);            \
            return SPOT_ERR_CUDA;                            \
        }                                                    \
    } while (0)

#define SPOT_LAUNCH_CHECK() SPOT_CUDA_TRY(cudaPeekAtLastError())

spot_status check_device();   // SPOT_ERR_UNSUPPORTED unless the current device is compute capability 10.x
int sm_count();

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: set it once per (kernel, device).  `done` is
// the call site's static bit mask of devices already configured.
template <typename F>
static inline cudaError_t set_max_smem_once(F kernel, int bytes, unsigned long long& done) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 64 && ((done >> dev) & 1ull)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && dev < 64) done |= 1ull << dev;
    return e;
}

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ---- quantised selector K-cache tile geometry (opaque layout, see include/spot.h) ------------------
// A tile holds SELK_TILE tokens: [SELK_TILE][H*d/2] code bytes, then [SELK_TILE][H*d/32] scale bytes.
// (f2: MXINT8 has H*d code bytes per token, INT4_BF16S two scale bytes per group -- selk_*_per_group below)
constexpr int SELK_TILE = 64;
__host__ __device__ constexpr bool selk_is_grouped(int fmt) {
    return fmt == SPOT_SELK_INT4_E4M3 || fmt == SPOT_SELK_MXFP4 || fmt == SPOT_SELK_MXINT8 || fmt == SPOT_SELK_INT4_BF16S;
}
__host__ __device__ constexpr bool selk_is_format(int fmt) { return fmt == SPOT_SELK_BF16 || fmt == SPOT_SELK_FP8_E4M3 || selk_is_grouped(fmt); }
__host__ __device__ constexpr int selk_code_bytes_per_group(int fmt) { return fmt == SPOT_SELK_MXINT8 ? 32 : 16; }
__host__ __device__ constexpr int selk_scale_bytes_per_group(int fmt) { return fmt == SPOT_SELK_INT4_BF16S ? 2 : 1; }
__host__ __device__ inline int64_t selk_codes_per_token(int H, int d) { return (int64_t)H * d / 2; }
__host__ __device__ inline int64_t selk_scales_per_token(int H, int d) { return (int64_t)H * d / 32; }
__host__ __device__ inline int64_t selk_tile_bytes(int H, int d) {
    return SELK_TILE * (selk_codes_per_token(H, d) + selk_scales_per_token(H, d));
}

// ---- pipelined decode step: cross-kernel hand-offs through global memory ---------------------------------------
// spot_select and spot_decode_step run score -> select (-> attend) as kernels that are resident TOGETHER: the scoring
// kernel walks the sequences in order on all of its CTAs; the selection CTA of a sequence waits for that sequence's block
// scores only, not for the end of the scoring grid, so the selection of sequence b overlaps the scoring of b + 1, ..; it
// then publishes ready[b], which is all an attention CTA waits for before it reads that sequence's index list.  Later
// kernels only ever wait on earlier ones (which are resident, or done, before a later one can start: programmatic
// dependent launch), never the other way round.
//
// No fence in the streaming kernel: a block score travels as ONE 64-bit word {tag, fp32 bits} (a naturally aligned
// 64-bit store is single-copy atomic), and the selection CTA simply re-reads an entry until it carries this call's tag
// -- a gpu-scope fence in a warp of the scoring kernel waits for the SM's bulk copies in flight (4-5 us each time,
// measured).  Only the selection kernel (one release per sequence) and the attention kernel (acquire loads) use
// ordered accesses.
//
// The words live in caller-owned workspace that need NOT be initialised: the tag is derived from a per-call token unlike
// the previous call's, and every reader clears what it has consumed (score tags: the selection CTA; ready words: the
// merge kernel, which runs when the attention grid has completed), so a finished call leaves no live tag behind -- which
// is what lets the replay of a captured graph (same token every time) start clean.
struct StepSync {
    uint32_t tag;                 // 0: no hand-offs (plain stream order through griddepcontrol.wait)
    uint32_t* ready;              // [B] == tag once the selection of sequence b is in global memory; nullptr: nobody waits
#ifdef SPOT_TRACE
    unsigned long long* trace;    // development builds only (-DSPOT_TRACE): [kernel][CTA < 512][4] %globaltimer stamps
#endif
};
static inline size_t step_sync_bytes(int B) { return (((size_t)B * 4 + 63) & ~(size_t)63); }

// ---- programmatic dependent launch (PDL) ------------------------------------------------------------
// The decode step is a chain of four short kernels (score -> select -> attend -> merge) whose launch latencies sit
// on the critical path.  Every kernel of the chain is launched with programmaticStreamSerializationAllowed = 1 and
//   * calls pdl_wait() before its first global read or write (returns once the previous kernel in the stream has
//     completed and its writes are visible; a no-op under an ordinary launch), on EVERY path, so that completion of
//     a kernel always implies completion of its predecessors;
//   * calls pdl_launch_dependents() right after, which lets the next kernel's CTAs become resident (and run their
//     own prologue up to pdl_wait()) as soon as SM resources allow.  All grids here fit on the chip in one wave, so
//     early-resident dependents never starve their predecessor.
#ifdef __CUDACC__
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                     Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif

// ---- device helpers ------------------------------------------------------------------------------
#ifdef __CUDACC__

__device__ __forceinline__ float bf16_bits_to_float(uint16_t b) { return __uint_as_float(((uint32_t)b) << 16); }
__device__ __forceinline__ float bf16lo(uint32_t v) { return __uint_as_float(v << 16); }
__device__ __forceinline__ float bf16hi(uint32_t v) { return __uint_as_float(v & 0xffff0000u); }

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&t);
}

// 128-bit streaming load (read-only path, no L1 allocation): the selector cache and KV are read once.
__device__ __forceinline__ uint4 ldg_stream_v4(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint2 ldg_stream_v2(const void* p) {
    uint2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
    return r;
}

// mma.sync m16n8k16, fp32 accumulate.  Used where M is tiny (decode: one query, or G <= 16 query heads);
// the dense prefill contraction uses tcgen05 instead (score_prefill.cu).
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma_f16_16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                              uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---- gpu-scope acquire / release on global words (the hand-offs of the pipelined decode step) --------------------
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(uint32_t* p, uint32_t v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add_u32(uint32_t* p, uint32_t v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
#ifdef SPOT_TRACE
__device__ __forceinline__ void trace_stamp(const StepSync& y, int kernel, int slot) {
    if (y.trace && threadIdx.x == 0 && blockIdx.x < 512) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        y.trace[((size_t)kernel * 512 + blockIdx.x) * 4 + slot] = t;
    }
}
#define SPOT_STAMP(y, k, slot) trace_stamp(y, k, slot)
#else
#define SPOT_STAMP(y, k, slot) ((void)0)
#endif

// one thread waits (with back-off) until *p == value
__device__ __forceinline__ void spin_until_eq(const uint32_t* p, uint32_t value) {
    while (ld_acquire_u32(p) != value) __nanosleep(64);
}
// tagged block scores (see StepSync): one 64-bit word {tag, fp32 bits}
__device__ __forceinline__ void st_tagged_score(unsigned long long* p, uint32_t tag, float s) {
    const unsigned long long v = ((unsigned long long)tag << 32) | (unsigned long long)__float_as_uint(s);
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_tagged_score(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// cp.async 16 B with zero-fill when !valid (src-size 0): out-of-range KV rows become zeros in smem.
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void* gptr, bool valid) {
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global.L2::128B [%0], [%1], 16, %2;" :: "r"(smem_addr), "l"(gptr), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

__device__ __forceinline__ void ldmatrix_x4(uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3, uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3, uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}

__device__ __forceinline__ float fast_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

#endif  // __CUDACC__

}  // namespace spot
