// Step a2 -- block distribution and selection rule, one CTA per selection row: reserved sink/recency
// tier, residual softmax (Eq. 7), nucleus + K_min floor (Eq. 8) or static top-K (Eq. 6).  This file marshals
// spot_select_params into the kernel's arguments; the kernel (histogram partition, rows of up to 2048 or 8192
// blocks) is in select_hist.cu.  (A bitonic-sort form -- 8 keys per thread, keys only, three strides per
// shared-memory round -- served rows of 2049..8192 blocks until the histogram kernel learned them: the decode step
// at 8192 blocks per row went from 168.9 to 158.8 us; it is gone.)
#include "select_common.cuh"

#include <string.h>

namespace spot {

spot_status launch_select_hist(const SelectArgs& a, int rows, int max_nb, cudaStream_t s);    // select_hist.cu

// sync (decode rows of a pipelined call): `scores` is then the scoring kernel's array of tagged 64-bit words, row stride
// nb_stride, and the plain block scores go to p->block_scores (row stride p->nb_stride) if the caller wants them.
spot_status run_select(const spot_select_params* p, const float* scores, int nb_stride, int rows_per_seq,
                       int max_nb, const StepSync* sync, cudaStream_t s) {
    if (max_nb > SEL_MAX_NB) return SPOT_ERR_UNSUPPORTED;
    SelectArgs a;
    memset(&a.sync, 0, sizeof(a.sync));
    a.tagged = nullptr; a.tagged_stride = 0; a.scores_out = nullptr; a.dry_from_row = 0;
    if (sync && sync->tag && p->q_block == 1) {
        a.sync = *sync;
        a.tagged = reinterpret_cast<unsigned long long*>(const_cast<float*>(scores));
        a.tagged_stride = nb_stride;
        a.scores_out = p->block_scores;
        scores = nullptr;
        nb_stride = p->nb_stride;              // rows of block_scores / block_probs
        // when do the scores of sequence b arrive?  ~4 us of ramp, then the cache streams at ~6.5 GB/ms; a dry pass
        // takes ~12 us, so only rows that arrive later than that gain from one
        const double bytes_per_seq = (double)p->max_seq_len * (double)spot_selector_k_bytes((spot_selk_format)p->fmt, 1, 64, p->H_idx, p->d_idx) / 64.0;
        // (the scoring grid walks the batch in min(B, 4) groups of consecutive sequences; a group's scores are complete
        // when the grid leaves it)
        const int n_groups = p->B < 4 ? p->B : 4;
        a.dry_from_row = p->B;
        for (int g = 0; g < n_groups; ++g) {
            const int b_end = (int)((long long)(g + 1) * p->B / n_groups);
            if (4.0 + b_end * bytes_per_seq / 6.5e6 >= 16.0) { a.dry_from_row = (int)((long long)g * p->B / n_groups); break; }
        }
    }
    a.scores = scores; a.nb_stride = nb_stride; a.seq_len = p->seq_len; a.max_len = p->max_seq_len; a.n_q = rows_per_seq;
    a.q_start = p->q_start; a.q_block = p->q_block; a.blk = p->blk;
    a.mode = p->mode; a.top_k = p->top_k; a.p = p->p; a.temperature = p->temperature;
    a.sink = p->sink_blocks; a.rec = p->recency_blocks; a.kmin = p->kmin_blocks;
    a.indices = p->indices; a.cap = p->cap; a.budgets = p->budgets; a.probs = p->block_probs;
    const int rows = p->B * rows_per_seq;
    return launch_select_hist(a, rows, max_nb, s);
}

}  // namespace spot
