/*
 * spot.h -- C ABI of the SpotAttention per-step hot path, B200 (sm_100a) build.
 *
 * The operations follow the paper's statement of the method (arxiv 2606.22874; cited below as
 * PAPER.md:<line> of the extracted text, plus the reading numbers R* of DESIGN.md section 3):
 *
 *   a0  spot_quantize_selector_k   group-32 "microscale" 4-bit selector K-cache
 *   a1  spot_select (scoring)      s_s[q,t] = sum_h w_h ReLU(q^I_h . k^I_{h,t})
 *                                  s_bar[q,b] = max_{t in b} s_s[q,t]
 *   a2  spot_select (selection)    static top-K (Eq. 6) or dual top-p: reserved sink/recency
 *                                  tier + nucleus on the residual softmax + K_min floor (Eq. 7-8)
 *   a3  spot_sparse_attn_decode    attention over the gathered K_I, V_I only           (PAPER.md:47 Fig. 2, :71)
 *   a3' spot_sparse_attn_prefill   the same under a causal mask, one index list per 64-token query block
 *
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless its name ends in _host.  The caller owns every buffer; the
 *     library never allocates, frees or keeps a pointer after the call returns.
 *   - Every call is asynchronous on the caller's stream (a cudaStream_t passed as void*; NULL = legacy
 *     default stream) and never synchronises.  All argument checks run on the host before any launch.
 *   - Device lengths are clamped: a seq_len[b] outside [0, max_seq_len] is read as the nearer bound (grids, score rows
 *     and workspaces are sized from max_seq_len, so a stale length cannot make a kernel leave its buffers).
 *   - Return value: spot_status.  SPOT_ERR_CUDA means a CUDA runtime call failed; the code is kept
 *     per thread and returned by spot_last_cuda_error().
 *   - BF16 tensors are passed as uint16_t bit patterns.  Pointers must be 16-byte aligned.
 *   - "block" = blk consecutive key tokens (the selection granularity): blk == 64 (BASELINE.json's configurations) or
 *     blk == 16 (the paper's own granularity) in every call, decode and prefill; a prefill query block is
 *     always 64 tokens.  A row may hold at most 8192 blocks (L <= 512K at blk 64, L <= 128K at blk 16).
 *   - No global state, no environment variables, no CPU fallback: on a device that is not compute
 *     capability 10.x every launching call returns SPOT_ERR_UNSUPPORTED.
 */
#ifndef SPOT_H_
#define SPOT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SPOT_OK = 0,
    SPOT_ERR_INVALID_ARG = 1,
    SPOT_ERR_UNSUPPORTED = 2,
    SPOT_ERR_WORKSPACE_TOO_SMALL = 3,
    SPOT_ERR_CUDA = 4
} spot_status;

/* Selector K-cache storage formats (R16/R17). */
typedef enum {
    SPOT_SELK_BF16 = 0,      /* [B][cache_stride_tokens][H_idx][d_idx] BF16                              */
    SPOT_SELK_INT4_E4M3 = 1, /* signed 4-bit codes, group 32 along d_idx, one FP8-E4M3 scale per group   */
    SPOT_SELK_MXFP4 = 2,     /* E2M1 codes, group 32 along d_idx, one E8M0 scale per group (OCP MX)      */
    SPOT_SELK_FP8_E4M3 = 3,  /* f2: one FP8-E4M3 byte per element, no scale, [B][tokens][H_idx][d_idx]   */
    SPOT_SELK_MXINT8 = 4,    /* f2: OCP MX INT8 codes (code * 2^-6), group 32, one E8M0 scale per group   */
    SPOT_SELK_INT4_BF16S = 5 /* f2: signed 4-bit codes, group 32, one BF16 scale per group: the paper's   */
                             /*     own INT4 accounting, 4.5 bit / element                 */
} spot_selk_format;

typedef enum {
    SPOT_MODE_TOPK = 0,      /* Eq. 6; K counts the reserved blocks (R10)                                */
    SPOT_MODE_DUAL_TOPP = 1  /* Eq. 7-8                                                                  */
} spot_select_mode;

const char* spot_status_string(spot_status s);
/* cudaError_t (as int) of the last failing CUDA call on this host thread; 0 if none. */
int spot_last_cuda_error(void);
/* Library version, "major.minor". */
const char* spot_version(void);
/* sizeof() of the parameter blocks as this library was compiled (which: 0 = spot_select_params,
 * 1 = spot_attn_params, 2 = spot_decode_step_host_params, 3 = spot_project_params, 4 = spot_decode_step_params,
 * 5 = spot_train_params; anything else: 0) -- lets a binding verify its layout. */
size_t spot_struct_size(int which);

/* ---------------------------------------------------------------------------------------------------
 * a0 -- selector K-cache formats.
 *
 * The quantised layout is OPAQUE: only spot_selector_k_bytes, spot_quantize_selector_k,
 * spot_dequantize_selector_k and spot_select define it.  (It is tiled by 64 tokens: the codes of a tile
 * followed by its scales, so that one tile is a single contiguous HBM stream.)
 *
 * Bytes of a cache holding B sequences of cache_stride_tokens tokens each (a multiple of 64 for the 4-bit
 * formats): BF16 2*n, 4-bit formats n/2 + n/32 with n = B*tokens*H_idx*d_idx (16 -> 4.25
 * bit/element), FP8-E4M3 n (the paper's "FP8" precision; R30: RNE-satfinite cast of every
 * element, no scale), MXINT8 n + n/32 (8.25 bit/element; R38), INT4 with a BF16 group scale n/2 + n/16
 * (PAPER.md:188's "4.5 bits per element", 1.27 GiB at Qwen3-8B / 128K; R39).  Returns 0 on invalid arguments.
 * --------------------------------------------------------------------------------------------------- */
size_t spot_selector_k_bytes(spot_selk_format fmt, int64_t B, int64_t cache_stride_tokens, int H_idx, int d_idx);

/* Quantise tokens [token_offset, token_offset + n_tokens) of every sequence.
 *   k_bf16   in   [B][n_tokens][H_idx][d_idx] BF16 (the new tokens only; dense)
 *   k_cache  out  cache in format fmt (SPOT_SELK_INT4_E4M3 or SPOT_SELK_MXFP4; SPOT_SELK_BF16 copies)
 * Prefill: the whole prompt; decode: n_tokens = 1 appended.  Requires d_idx % 32 == 0,
 * token_offset + n_tokens <= cache_stride_tokens.  Quantiser definitions: DESIGN.md R16 (MXFP4: scale
 * 2^(floor(log2 amax) - 2), RNE onto the E2M1 grid, saturating; INT4: scale = E4M3_rne_satfinite(amax/7),
 * q = clamp(rint(v/scale), -7, 7)); R38 (MXINT8: scale 2^floor(log2 amax), code = clamp(RNE(64 v / scale), -127, 127));
 * R39 (INT4_BF16S: scale = RNE_bf16(amax/7), q as INT4).  Results are bit-exact with that definition. */
spot_status spot_quantize_selector_k(const uint16_t* k_bf16, void* k_cache, spot_selk_format fmt,
                                     int64_t B, int64_t n_tokens, int64_t token_offset,
                                     int64_t cache_stride_tokens, int H_idx, int d_idx, void* stream);

/* Inverse: write the dequantised keys of tokens [token_offset, token_offset + n_tokens) as BF16
 * [B][n_tokens][H_idx][d_idx] (exact: every dequantised value is representable in BF16 -- except SPOT_SELK_INT4_BF16S,
 * whose values q * scale carry up to 11 significant bits: for that format this call writes their round-to-nearest-even
 * BF16 view, a diagnostic; the scoring kernels use the exact products, and prefill selection (q_block = 64), which would
 * go through this view, returns SPOT_ERR_UNSUPPORTED). */
spot_status spot_dequantize_selector_k(const void* k_cache, uint16_t* k_bf16_out, spot_selk_format fmt,
                                       int64_t B, int64_t n_tokens, int64_t token_offset,
                                       int64_t cache_stride_tokens, int H_idx, int d_idx, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * f1 -- the step right before the path (decode form): selector projections, RoPE, mixing weights, and the
 * append of the new token's selector key to the (quantised) cache, PAPER.md:39 ("q^I_h, k^I_{h,t} are the
 * per-head query/key projections and W_w a small linear map producing the per-query mixing weights w_h from
 * the hidden state h_q"), PAPER.md:362-364 (4 heads, "RoPE head dim 64").  Readings R27-R29 of DESIGN.md:
 *   q^I = W_q h, k^I = W_k h, w = W_w h (no bias, no activation; BF16 inputs, fp32 accumulation);
 *   rotary embedding on the first rope_dims dims of every selector head of q^I and k^I, rotate-half pairing
 *   (i, i + rope_dims/2), angle = pos * rope_base^(-2 i / rope_dims); the other dims pass through;
 *   q^I and k^I are rounded once to BF16 after the rotation; the cache entry of token pos[b] of sequence b is
 *   that BF16 k^I in format fmt (quantised exactly as spot_quantize_selector_k would quantise it).
 * One token per sequence.  A sequence whose pos[b] lies outside [0, cache_stride_tokens) gets sel_q and w but no
 * cache write.  Requires d_model % 256 == 0, d_idx % 32 == 0, rope_dims even and <= d_idx, H_idx * d_idx % 2 == 0.
 * workspace: >= spot_selector_project_append_workspace_bytes (the BF16 k^I of the new tokens, B * H_idx * d_idx * 2).
 * --------------------------------------------------------------------------------------------------- */
typedef struct {
    const uint16_t* hidden;      /* [B][d_model] BF16 hidden state h of the current token                */
    const uint16_t* w_q;         /* [H_idx*d_idx][d_model] BF16, row r = head r / d_idx, dim r % d_idx   */
    const uint16_t* w_k;         /* [H_idx*d_idx][d_model] BF16                                           */
    const uint16_t* w_w;         /* [H_idx][d_model] BF16                                                 */
    const int32_t* pos;          /* [B] device: absolute position of the token = its slot in the cache    */
    int32_t B, d_model, H_idx, d_idx, rope_dims;
    float rope_base;
    uint16_t* sel_q;             /* out [B][H_idx][d_idx] BF16                                            */
    float* w;                    /* out [B][H_idx] fp32                                                   */
    void* sel_k;                 /* selector K-cache, format fmt                                          */
    int32_t fmt;                 /* spot_selk_format                                                      */
    int64_t cache_stride_tokens;
    void* workspace;
    size_t workspace_bytes;
} spot_project_params;

size_t spot_selector_project_append_workspace_bytes(const spot_project_params* p);
spot_status spot_selector_project_append(const spot_project_params* p, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * a1 + a2 -- spot_select: scores, block distribution, selection, index list + per-query budget.
 *
 * Rows.  The call handles B sequences x n_q selection rows each:
 *   decode  (q_block == 1, Tq == 1): n_q = 1; the query sits at position seq_len[b]-1 and sees keys
 *           0..seq_len[b]-1 (the current token is already appended, R15); n_b = ceil(seq_len[b]/blk).
 *   prefill (q_block == 64): Tq % 64 == 0, n_q = Tq/64; query block i covers absolute positions
 *           [q_start + 64 i, q_start + 64 i + 64); it sees key blocks 0..n_b(i)-1 with n_b(i) the index
 *           of the block holding its last token, plus one; one tile score per (query block, key block) =
 *           max over the block's queries and the block's causally visible keys (R2).
 * Reserved tier: the first sink_blocks and the last recency_blocks of the row's n_b blocks.
 * Dual top-p (Eq. 7-8): p~ = softmax over the residual blocks of s_bar/temperature; nucleus = shortest
 * prefix in (score descending, index ascending) order whose mass is >= p (p >= 1: all residual blocks);
 * then extended in the same order until the budget reaches min(kmin_blocks, n_b).  Top-K (Eq. 6):
 * reserved plus the max(0, top_k - |reserved|) best residual blocks.
 *
 * Outputs (row r = b*n_q + i):
 *   indices      int32 [B*n_q][cap]   selected block ids, ascending, padded with -1
 *   budgets      int32 [B*n_q]        |S_q| including the reserved blocks
 *   block_scores fp32  [B*n_q][nb_stride]  optional (may be NULL): s_bar; entries >= n_b(row) undefined
 *   block_probs  fp32  [B*n_q][nb_stride]  optional: p~ on the residual blocks, 0 on reserved ones
 * cap must be >= the largest budget any row can reach (>= min(n_b, what the mode allows)); a row whose
 * budget would exceed cap makes the call fail up front when detectable on the host (cap < max n_b for
 * DUAL_TOPP, cap < min(top_k, max n_b) for TOPK) with SPOT_ERR_INVALID_ARG.
 *
 * Supported selector geometries: H_idx == 4 with d_idx == 64 or 128 (anything else: SPOT_ERR_UNSUPPORTED), every cache
 * format in both row forms.  Prefill rows over a quantised cache dequantise the visible prefix into the workspace
 * first (spot_select_workspace_bytes accounts for it) -- unless the queries are quantised too (q_fmt below).
 * --------------------------------------------------------------------------------------------------- */
typedef struct {
    /* inputs */
    const uint16_t* sel_q;       /* [B][Tq][H_idx][d_idx] BF16 selector queries q^I                       */
    const float* w;              /* [B][Tq][H_idx] fp32 mixing weights w_h (any sign, R13)               */
    const void* sel_k;           /* selector K-cache, format fmt                                          */
    int32_t fmt;                 /* spot_selk_format                                                      */
    int64_t cache_stride_tokens; /* tokens of capacity per sequence in sel_k                              */
    const int32_t* seq_len;      /* [B] device; decode: valid tokens per sequence (>= 1).  prefill: NULL  */
    int32_t max_seq_len;         /* host-side upper bound of seq_len (decode) -- sizes the grid           */
    int32_t B, Tq, H_idx, d_idx;
    int32_t q_start;             /* prefill: absolute position of the first query (multiple of 64)        */
    int32_t blk;                 /* key block size: 64 or 16                                              */
    int32_t q_block;             /* 1 = decode form, 64 = prefill form                                    */
    /* rule */
    int32_t mode;                /* spot_select_mode                                                      */
    int32_t top_k;
    double p;                    /* in (0, 1]; fp64 so that the mass threshold is the caller's exact value */
    int32_t sink_blocks, recency_blocks, kmin_blocks;
    double temperature;          /* > 0 (default 1.0)                                       */
    /* outputs */
    int32_t* indices;
    int32_t cap;
    int32_t* budgets;
    float* block_scores;         /* optional */
    float* block_probs;          /* optional */
    int32_t nb_stride;           /* row stride (elements) of block_scores / block_probs; >= max n_b       */
    /* scratch */
    void* workspace;
    size_t workspace_bytes;      /* >= spot_select_workspace_bytes(&params)                               */
    /* f2 -- quantised selector QUERIES on the tensor cores ("queries and key cache").  0 (SPOT_SELK_BF16,
     * the default): sel_q is BF16.  SPOT_SELK_FP8_E4M3: sel_q is FP8-E4M3 bytes [B][Tq][H_idx][d_idx] (what
     * spot_quantize_selector_k writes for a cache of Tq tokens), accepted with fmt == SPOT_SELK_FP8_E4M3 and q_block == 64
     * only (SPOT_ERR_UNSUPPORTED otherwise): the tile scores are then FP8 x FP8 products accumulated in fp32 by
     * tcgen05.mma kind::f8f6f4 straight from the cache -- no dequantise pass, no BF16 scratch.  The result is the score of
     * the two dequantised images (R33).  SPOT_SELK_MXFP4: sel_q is an MXFP4 cache of Tq tokens per sequence
     * (spot_quantize_selector_k with cache_stride_tokens = Tq; spot_selector_k_bytes(MXFP4, B, Tq, ..) bytes), accepted
     * with fmt == SPOT_SELK_MXFP4 and q_block == 64 only: E2M1 x E2M1 products times the two groups' UE8M0 scales,
     * accumulated in fp32 by tcgen05.mma kind::mxf4.block_scale (group scales through tensor memory), again straight from
     * the opaque cache layout and with the score of the two dequantised images as the result. */
    int32_t q_fmt;
} spot_select_params;

size_t spot_select_workspace_bytes(const spot_select_params* p);
spot_status spot_select(const spot_select_params* p, void* stream);

/* a1 / a1' alone -- the scoring half of spot_select: writes s_bar into block_scores (required,
 * row stride nb_stride) and stops; the rule fields, indices, budgets, cap and the workspace are ignored.  Same
 * argument checks and errors as spot_select otherwise (one exception: prefill rows over a quantised cache need
 * spot_select_workspace_bytes of workspace for the dequantised prefix).  Lets a caller (and bench.py) run and time the selector
 * scoring kernel by itself. */
spot_status spot_score_blocks(const spot_select_params* p, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * a3 / a3' -- block-sparse GQA attention over the selected KV blocks.
 *
 *   o_h = sum_{t in T_q} softmax_t(sm_scale * q_h . k_{g,t}) v_{g,t},  g = floor(h / (H_q/H_kv)),
 *   T_q = tokens of the selected blocks that are valid (t < seq_len[b]; prefill: t <= own position).
 * One index list per (sequence, query row) shared by all heads (R14).  K and V are BF16 with D = 128
 * contiguous and element strides for batch / token / head, so both [B][L][H_kv][D] and [B][H_kv][L][D]
 * work.  fp32 softmax and accumulation, BF16 output.
 *
 * decode:  q [B][H_q][D], one row per sequence; indices [B][cap], budgets [B].
 * prefill: q [B][Tq][H_q][D] at absolute positions q_start.., Tq % 64 == 0, q_start % 64 == 0;
 *          indices [B*Tq/64][cap], budgets [B*Tq/64]; seq_len unused (keys up to q_start+Tq-1 must exist).
 * indices == NULL means "every block" (the dense comparator); budgets is then ignored.
 * lse (optional, fp32 [B][H_q] decode / [B][Tq][H_q] prefill): natural-log sum-exp of the scaled logits.
 * Requires H_q % H_kv == 0, H_q/H_kv <= 16, D == 128, blk == 64 or 16 (prefill with blk == 16: a list entry is a
 * 16-token block; a query token attends to the entry's tokens at or before its own position, so an entry may be wholly
 * invisible to the first rows of the query block that selected it).
 * --------------------------------------------------------------------------------------------------- */
typedef struct {
    const uint16_t* q;
    const uint16_t* k;
    const uint16_t* v;
    int64_t kv_stride_batch, kv_stride_token, kv_stride_head; /* in elements */
    const int32_t* seq_len;      /* [B] device (decode) */
    int32_t max_seq_len;         /* host upper bound of seq_len (decode; sizes the dense grid)            */
    const int32_t* indices;
    const int32_t* budgets;
    int32_t cap;                 /* row stride of indices                                                 */
    int32_t B, Tq, H_q, H_kv, D;
    int32_t q_start;
    int32_t blk;
    float sm_scale;
    uint16_t* out;               /* BF16, same shape as q                                                 */
    float* lse;                  /* optional                                                              */
    void* workspace;
    size_t workspace_bytes;
    /* Paged K/V (f3, R32).  page_table == NULL: contiguous caches as described above.
     * Otherwise k and v are page POOLS: logical token t of sequence b is row t % page_tokens of physical page
     * page_table[b * page_table_stride + t / page_tokens]; kv_stride_batch is then the element stride between
     * PAGES (a multiple of kv_stride_token), kv_stride_token / kv_stride_head apply inside a page.  page_tokens is a
     * multiple of 16 (prefill: of 64, a key block must sit inside one page; SPOT_ERR_UNSUPPORTED otherwise).  Entries
     * for logical pages at or past ceil(seq_len[b] / page_tokens) (prefill: past q_start + Tq) are never read.  Page
     * numbers are < 2^22. */
    const int32_t* page_table;   /* device, int32 [B][page_table_stride]                                  */
    int32_t page_table_stride;
    int32_t page_tokens;
} spot_attn_params;

size_t spot_sparse_attn_decode_workspace_bytes(const spot_attn_params* p);
spot_status spot_sparse_attn_decode(const spot_attn_params* p, void* stream);

/* spot_sparse_attn_decode for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same operation, arguments, checks, launches and results (bit for bit), but the split-KV
 * partials live in an array INSIDE the library (a file-scope `static __device__` array of SPOT_STATIC_SCRATCH_BYTES,
 * held by every GPU that loads the library until the process exits).  p->workspace / p->workspace_bytes are ignored
 * (may be NULL / 0); inputs and outputs are the caller's as before.  The call allocates nothing and frees nothing.
 *   - Limit: spot_sparse_attn_decode_workspace_bytes(p) <= SPOT_STATIC_SCRATCH_BYTES, i.e.
 *     2 * (2 * SM count + B * H_kv) * (H_q / H_kv) * 520 bytes (B = 16, H_kv = 8, H_q / H_kv = 4 on a B200: 1.7 MiB; H_q / H_kv = 16,
 *     B * H_kv <= 208 fits).  A larger problem is refused with SPOT_ERR_WORKSPACE_TOO_SMALL before anything is launched:
 *     use spot_sparse_attn_decode with a workspace of your own.
 *   - ONE array per GPU, shared by every call: calls that overlap on the GPU (two streams, two host threads on one
 *     device) RACE on it -- serialise them, or use the workspace form.  Calls on one stream are ordered and safe.
 *   - The array keeps the previous call's contents; nothing in it has to start at zero (every partial the merge reads
 *     is written by the same call first), so there is no clearing pass. */
#define SPOT_STATIC_SCRATCH_BYTES (8u << 20)
spot_status spot_sparse_attn_decode_static(const spot_attn_params* p, void* stream);

size_t spot_sparse_attn_prefill_workspace_bytes(const spot_attn_params* p);
spot_status spot_sparse_attn_prefill(const spot_attn_params* p, void* stream);

/* Bench-only comparator: dense flash-decode of the same shapes (every block, no index list).  Same
 * parameter block; indices / budgets are ignored. */
size_t spot_dense_attn_decode_workspace_bytes(const spot_attn_params* p);
spot_status spot_dense_attn_decode(const spot_attn_params* p, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * One decode layer-step in ONE call: a1 + a2 + a3 (spot_select followed by spot_sparse_attn_decode over the lists it
 * wrote), same arithmetic, same outputs, same parameter blocks -- but launched as kernels that overlap (DESIGN.md
 * section 7): the scoring kernel walks the sequences in order, the selection of sequence b runs (on SMs left to it) while
 * sequences b + 1.. are still being scored, and the attention kernel, resident as soon as the scoring CTAs retire,
 * starts on the sequences whose lists are ready and takes the last sequence last, so that no selection latency sits
 * between the two HBM streams.  The hand-offs are a few words in `workspace` (flags and counters; the workspace need not
 * be initialised and may be reused by the next call on the same stream; two calls in flight on different streams need
 * two workspaces).
 *   select / attn: as for the separate calls, with the SAME indices / budgets / cap / seq_len / max_seq_len / blk / B in
 *   both (SPOT_ERR_INVALID_ARG otherwise), q_block == 1; each still carries its own workspace.
 * Like every call: asynchronous on `stream`, never synchronises, capturable in a CUDA graph.
 * --------------------------------------------------------------------------------------------------- */
typedef struct {
    spot_select_params select;
    spot_attn_params attn;
    void* workspace;
    size_t workspace_bytes;      /* >= spot_decode_step_workspace_bytes(&params)                          */
} spot_decode_step_params;

size_t spot_decode_step_workspace_bytes(const spot_decode_step_params* p);
spot_status spot_decode_step(const spot_decode_step_params* p, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * Host-buffer convenience (the "e2e" path of bench.py): one decode layer-step with every per-step tensor in HOST
 * memory.  Copies the step's inputs host->device into caller-provided device staging buffers, runs spot_decode_step,
 * copies the attention output and the budgets back (the index lists stay on the device: `out | budgets` is all that
 * returns), all on `stream`, no sync.
 * The *_host buffers must be PAGE-LOCKED (cudaHostAlloc / cudaHostRegister; SPOT_ERR_INVALID_ARG otherwise): a copy from
 * pageable memory would block the host and could not be captured.  Every argument check runs before the first copy.
 * When the host inputs are laid out back to back (sel_q | w | q) and so are their device staging areas, they go up as
 * ONE transfer; likewise out | budgets come back as one (each small copy costs microseconds of stream time).
 * (Declared here so that the end-to-end measurement also crosses the C ABI.)
 * --------------------------------------------------------------------------------------------------- */
typedef struct {
    /* host inputs for this step */
    const uint16_t* sel_q_host;  /* [B][H_idx][d_idx] */
    const float* w_host;         /* [B][H_idx] */
    const uint16_t* q_host;      /* [B][H_q][D] */
    /* host outputs */
    uint16_t* out_host;          /* [B][H_q][D] */
    int32_t* budgets_host;       /* [B] */
    /* device-resident state and staging; select/attn hold the device pointers of everything else */
    spot_select_params select;   /* sel_q / w point at device staging */
    spot_attn_params attn;       /* q / out point at device staging   */
    void* step_workspace;        /* device, >= spot_decode_step_workspace_bytes of the same select / attn  */
    size_t step_workspace_bytes;
} spot_decode_step_host_params;

spot_status spot_decode_step_host(const spot_decode_step_host_params* p, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * f4 -- the training-side reductions of ONE sequence (the other half of the method), on synthetic or real
 * tensors alike; no L x L matrix is stored.
 *   teacher  p^tau[q,t]   = (1/H_q) sum_h softmax_t(sm_scale q_h . k_{g(h),t})  over t <= q   (Eq. 1: softmax, then mean)
 *   student  p^sigma[q,t] = softmax_t(s_s[q,t]) over t <= q, s_s as in spot_select              (Eq. 2)
 *   dense_kl[q]  = sum_t p^tau log(p^tau / p^sigma)                                             (Eq. 3; the loss is its mean)
 *   sparse_kl[q] = the same over S_q with both distributions renormalised there                 (Eq. 4)
 * S_q (R35) = the tokens t <= q of the top_k best key blocks of query q by block-max score -- Eq. 6 applied per
 * query, reserved sink / recency blocks counted inside top_k as in spot_select; the paper's K_train = 8192 tokens at
 * blk = 16 is top_k = 512.  0 log 0 = 0; a query whose S_q carries no teacher mass gets 0.
 *   q      [L][H_q][D] BF16          k  BF16 with element strides (token, head), D contiguous (no V: nothing here needs it)
 *   sel_q  [L][H_idx][d_idx] BF16    w  [L][H_idx] fp32      sel_k  [L][H_idx][d_idx] BF16 (the BF16 cache layout)
 *   dense_kl, sparse_kl  out fp32 [L];  teacher_lse  optional out fp32 [L][H_q], natural-log sum-exp of the scaled logits
 *   indices / budgets    optional out (both or neither): the block lists of S_q, int32 [L][cap] ascending, -1 padded, and
 *                        their lengths; cap >= min(top_k, ceil(L / blk))
 * Requires D == 128, H_kv <= 8, H_q / H_kv in {2, 4, 8, 16}, H_idx <= 4, d_idx % 16 == 0 and <= 128, blk in {16, 32, 64},
 * ceil(L / blk) <= 8192 (SPOT_ERR_UNSUPPORTED otherwise).  fp32 softmax statistics and sums; the logits are exact BF16
 * products accumulated in fp32.
 * --------------------------------------------------------------------------------------------------- */
typedef struct {
    const uint16_t* q;
    const uint16_t* k;
    int64_t k_stride_token, k_stride_head;   /* in elements */
    const uint16_t* sel_q;
    const float* w;
    const uint16_t* sel_k;
    int32_t L, H_q, H_kv, D, H_idx, d_idx;
    int32_t blk, top_k, sink_blocks, recency_blocks;
    float sm_scale;
    float* dense_kl;
    float* sparse_kl;
    float* teacher_lse;          /* optional */
    int32_t* indices;            /* optional */
    int32_t* budgets;            /* optional */
    int32_t cap;
    void* workspace;
    size_t workspace_bytes;      /* >= spot_train_kl_workspace_bytes(&params)                             */
} spot_train_params;

size_t spot_train_kl_workspace_bytes(const spot_train_params* p);
spot_status spot_train_kl(const spot_train_params* p, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* SPOT_H_ */
