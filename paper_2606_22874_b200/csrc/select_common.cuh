// Shared by select.cu (argument marshalling) and select_hist.cu (the selection kernel).
#pragma once
#include "common.cuh"

namespace spot {

constexpr int SEL_MAX_NB = 8192;
constexpr uint32_t KEY_PAD = 0xffffffffu;

__device__ __forceinline__ uint32_t orderable(float x) {
    uint32_t u = __float_as_uint(x + 0.0f);   // -0.0 -> +0.0
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float from_orderable(uint32_t o) {
    uint32_t u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
    return __uint_as_float(u);
}
// sort key: ascending key == descending score
__device__ __forceinline__ uint32_t score_key(float s) { return ~orderable(s); }
__device__ __forceinline__ float key_score(uint32_t k) { return from_orderable(~k); }

struct SelectArgs {
    const float* scores;      // [rows][nb_stride]
    int nb_stride;
    const int32_t* seq_len;   // decode: [B]; prefill: nullptr
    int max_len;              // decode: host-side bound of seq_len (device values are clamped to [0, max_len])
    int n_q;                  // rows per sequence
    int q_start, q_block, blk;
    int mode, top_k;
    double p, temperature;
    int sink, rec, kmin;
    int32_t* indices;
    int cap;
    int32_t* budgets;
    float* probs;             // optional [rows][nb_stride]
    StepSync sync;            // pipelined step (decode rows): publish ready[b]; tag == 0: plain stream order
    unsigned long long* tagged;   // pipelined step: the scoring kernel's {tag, fp32 bits} words [rows][tagged_stride] (read
    int tagged_stride;            //   until tagged, then cleared); block scores are copied to scores_out when it is set
    float* scores_out;            // [rows][nb_stride] or nullptr
    int dry_from_row;             // pipelined step: sequences >= this one warm the kernel's code with a dry pass first
};

}  // namespace spot
