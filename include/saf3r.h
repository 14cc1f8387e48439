/*
 * saf3r.h -- C ABI of the B200-native (sm_100a) SAF3R hot path.
 *
 * The hot path is the per-head dynamic sparse cross-view global attention of SAF3R
 * (arxiv/paper_2607_03612; line numbers below are /root/reference/PAPER.md):
 *   step 1  saf3r_select      -- online pattern adaptation (Sec. 4.3) restated at token-block
 *                                granularity: pool Q/K into blocks, score block pairs, select a per-head block mask
 *                                according to the head's type (Sec. 4.1).
 *   step 2  saf3r_sparse_attn -- block-sparse softmax attention over the selected K/V blocks.
 *   dense   saf3r_dense_attn  -- O_full = softmax(QK^T/sqrt(D))V, the library's own speedup baseline.
 *
 * Conventions
 *   - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. torch tensors); pointers named *_host are
 *     plain host memory.  The library allocates no device memory after saf3r_create.
 *   - q, k, v, out: bf16 (out optionally fp32), logical layout [H][N][D] addressed through two element strides
 *     (stride_head, stride_token); the head_dim stride is 1.  N = num_frames * tokens_per_frame.
 *     q/k/v base pointers must be 16-byte aligned and both strides multiples of 8 elements (TMA requirement).
 *   - Token t belongs to frame floor(t/T) at in-frame position t mod T; block J holds tokens [J*B, min((J+1)*B, N)).
 *   - Asynchrony: select / *_attn enqueue work on `cuda_stream` (a cudaStream_t passed as void*) and return.
 *     Argument errors are returned synchronously before anything is enqueued.
 *   - Errors: every call returns a saf3r_status; text via saf3r_last_error(ctx).  SAF3R_ERR_CUDA is sticky.
 *   - A context is not thread-safe: use one context per host thread (or serialise calls).  Calls on one context may target
 *     different streams one after another; saf3r_layer_host additionally uses context-owned side streams.
 *   - Attention calls in flight per context: every *_attn call takes the next of 256 context-owned slots (per-head key-norm
 *     bounds and the head order its kernel reads) and the slot is reused, without any wait, 256 attention calls later.  Keep
 *     fewer than 256 attention calls of one context unfinished at a time.  A CUDA graph captured from such calls (e.g. the stack
 *     of paper_2607_03612_b200/stack.py) has its slots baked in: while a replay of it may be running, do not issue 256 or more
 *     eager attention calls on the same context from another stream (they would wrap the ring and overwrite the replay's slots,
 *     which can freeze the running max too early and yield inf/NaN) - use a second context for that stream.
 *   - There is no CPU fallback: on a machine without an sm_100 device saf3r_create fails with SAF3R_ERR_UNSUPPORTED.
 */
#ifndef SAF3R_H_
#define SAF3R_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#ifndef SAF3R_MAX_HEADS
#define SAF3R_MAX_HEADS 64 /* per call; a batch folds into the head dimension */
#endif

typedef struct saf3r_ctx saf3r_ctx; /* opaque; owns its tensor-map cache, a tiny device scratch and the error string */

typedef enum {
  SAF3R_OK = 0,
  SAF3R_ERR_INVALID_ARG = 1,
  SAF3R_ERR_UNSUPPORTED = 2, /* head_dim != 64, block not in {64,128}, H > SAF3R_MAX_HEADS, non-sm_100 device */
  SAF3R_ERR_CAPACITY = 3,    /* lists / workspace buffer too small (required sizes: saf3r_query_sizes) */
  SAF3R_ERR_CUDA = 4
} saf3r_status;

/* Head types = the paper's four tailored kernels + dense. */
typedef enum {
  SAF3R_HEAD_DENSE = 0,            /* all k-blocks (O_full) */
  SAF3R_HEAD_UNIFORM_STRIDE = 1,   /* "Uniform Sampling Kernel", PAPER.md:L102 (scanning heads; also c_base, L106) */
  SAF3R_HEAD_STATIC = 2,           /* "Static Kernel", PAPER.md:L96 (position heads) */
  SAF3R_HEAD_QUERY_PROBE_TOPK = 3, /* "Query-Probe Top-K Kernel", PAPER.md:L98, L122-124 (vertical-line heads) */
  SAF3R_HEAD_BLOCK_TOPK = 4,       /* block-wise similarity Top-K, PAPER.md:L100, L126 (correspondence heads) */
  SAF3R_HEAD_CACHED = 5            /* reuse the lists of head `offset` of an index cache computed once per sequence
                                      ("the indices are cached and reused by all subsequent ... kernels");
                                      only valid in saf3r_select_cached */
} saf3r_head_type;
typedef enum { SAF3R_STATIC_ANCHOR = 0, SAF3R_STATIC_FRAME_LOCAL = 1, SAF3R_STATIC_POSITION_BAND = 2 } saf3r_static_mode;
typedef enum { SAF3R_SCOPE_GLOBAL = 0, SAF3R_SCOPE_PER_FRAME = 1 } saf3r_topk_scope;
typedef enum { SAF3R_SCORE_DOT = 0, SAF3R_SCORE_COSINE = 1 } saf3r_score_mode;

/* One per head; plain host memory; all fields int32.  Selection rules (list of q-block I, ascending k-block indices):
 *   DENSE            {0..NB-1}
 *   UNIFORM_STRIDE   stride>=1: {offset + i*stride < NB} (0 <= offset < stride);  stride==0: {floor(i*NB/keep_blocks)}
 *   STATIC/ANCHOR    blocks covering frame `anchor_frame`
 *   STATIC/FRAME_LOCAL  blocks covering the frame(s) the tokens of q-block I belong to
 *   STATIC/POSITION_BAND  for the in-frame positions [pa,pb] of q-block I: blocks covering positions
 *                    [max(0,pa-r), min(T-1,pb+r)] of EVERY frame, r = band_radius
 *   QUERY_PROBE_TOPK top-`keep_blocks` of p[J] = qbar . Ktilde_J / sqrt(D), same list for every I
 *   BLOCK_TOPK       s[I][J] = Qtilde_I . Ktilde_J * c (c = 1/sqrt(D) for DOT; COSINE pools L2-normalised tokens, c = 1);
 *                    GLOBAL: top-`keep_blocks` of the row; PER_FRAME: top-`topk_per_frame` inside each frame's
 *                    candidate blocks {J : floor(J*B/T) = g}, union over frames g.
 *   CACHED           the rows of head `offset` of the cache passed to saf3r_select_cached, copied; keep_blocks / topk_scope /
 *                    topk_per_frame must repeat the rule the cache head was built with (they fix the list lengths)
 *   Top-n uses the total order (score descending, then index ascending). */
typedef struct {
  int32_t type;
  int32_t stride, offset;
  int32_t keep_blocks;
  int32_t static_mode, anchor_frame, band_radius;
  int32_t topk_scope, topk_per_frame;
  int32_t score_mode;
} saf3r_head_cfg;

typedef struct {
  int32_t num_frames, tokens_per_frame, num_heads, head_dim, block;
  int64_t stride_head, stride_token; /* element strides of q/k/v/out */
} saf3r_shape;

/* CSR block lists: list of (h, I) = col_idx[row_ptr[h*NB+I] .. row_ptr[h*NB+I+1]), ascending, unique, 0 <= J < NB.
 * An open format: callers may pass hand-made lists to saf3r_sparse_attn.  An empty list yields zero output rows
 * and lse = -inf. */
typedef struct {
  int64_t *row_ptr; /* dev, [H*NB + 1] */
  int32_t *col_idx; /* dev */
  int64_t capacity; /* entries available in col_idx */
} saf3r_lists;

/* Create a context on CUDA device `device` (must be sm_100).  Returns SAF3R_ERR_UNSUPPORTED otherwise. */
saf3r_status saf3r_create(saf3r_ctx **ctx, int device);
void saf3r_destroy(saf3r_ctx *ctx);
const char *saf3r_last_error(const saf3r_ctx *ctx);

/* Host-only sizing.  List lengths are a closed form of (shape, cfg) for every head type, never of the data.
 * list_entries: total col_idx entries saf3r_select will write.  workspace_bytes: device scratch saf3r_select needs
 * (pooled Qtilde/Ktilde fp32, qbar, row lengths). cfg: host array [H]. */
saf3r_status saf3r_query_sizes(const saf3r_shape *shape, const saf3r_head_cfg *cfg_host, int64_t *list_entries,
                               size_t *workspace_bytes);

/* Step 1: pool -> score -> select.  Writes out_lists->row_ptr (all H*NB+1 entries) and col_idx.
 * SAF3R_ERR_CAPACITY if out_lists->capacity or workspace_bytes is too small. */
saf3r_status saf3r_select(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const saf3r_shape *shape,
                          const saf3r_head_cfg *cfg_host, void *workspace_dev, size_t workspace_bytes,
                          saf3r_lists *out_lists, void *cuda_stream);

/* Step 1 with an index cache: `cache` holds the lists of `cache_heads` BLOCK_TOPK heads
 * computed ONCE per sequence by an ordinary saf3r_select call on a caller-supplied feature tensor (q = k = features,
 * SAF3R_SCORE_COSINE reproduces the paper's cosine similarity of patch features at block level).  Heads of type
 * SAF3R_HEAD_CACHED copy their rows from cache head `offset`; all other heads behave as in saf3r_select, so a layer whose
 * correspondence heads are CACHED pools and scores only for its QUERY_PROBE heads.  The cache must have been built for the
 * same (num_frames, tokens_per_frame, block); it is only read.  cache == NULL makes this identical to saf3r_select. */
saf3r_status saf3r_select_cached(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const saf3r_shape *shape,
                                 const saf3r_head_cfg *cfg_host, const saf3r_lists *cache, int32_t cache_heads,
                                 void *workspace_dev, size_t workspace_bytes, saf3r_lists *out_lists, void *cuda_stream);

/* Step 2: o_i = sum_j softmax_j(q_i.k_j/sqrt(D)) v_j over j in the blocks of list(h, blk(i)), j < N.
 * out_dev: bf16 (out_is_fp32 = 0) or fp32 (1), same [H][N][D] strides as q.  lse_dev_or_null: fp32 [H][N] contiguous,
 * natural-log log-sum-exp of the kept logits. */
saf3r_status saf3r_sparse_attn(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const void *v_dev,
                               const saf3r_shape *shape, const saf3r_lists *lists, void *out_dev, int out_is_fp32,
                               float *lse_dev_or_null, void *cuda_stream);

/* Validates caller-made lists (the format is open): row_ptr non-decreasing and within capacity, every row ascending, unique and
 * inside [0, NB).  Writes the number of malformed rows to *bad_rows_host.  Synchronises `cuda_stream` (a debugging aid, not
 * part of the hot path; saf3r_sparse_attn itself does not validate). */
saf3r_status saf3r_check_lists(saf3r_ctx *ctx, const saf3r_shape *shape, const saf3r_lists *lists, int64_t *bad_rows_host,
                               void *cuda_stream);

/* Union of two sets of block lists, row by row ("combining Top-K with uniform striding to
 * reduce missing regions"): out(h, I) = a(h, I) U b(h, I), ascending and unique - e.g. the lists of one saf3r_select call with
 * BLOCK_TOPK rules and of another with UNIFORM_STRIDE rules.  a, b: lists over the same (H, NB); out: caller-owned, must not
 * alias an input; out->capacity >= entries(a) + entries(b) always suffices.  Entries that would not fit out->capacity are not
 * written; out->row_ptr[H*NB] always holds the true total, so a caller in doubt compares it with the capacity
 * (saf3r_check_lists reports such lists as malformed).  Three launches (count, scan, write); enqueues and returns. */
saf3r_status saf3r_union_lists(saf3r_ctx *ctx, const saf3r_shape *shape, const saf3r_lists *a, const saf3r_lists *b,
                               saf3r_lists *out, void *cuda_stream);

/* Dense mode of the same kernel (implicit list 0..NB-1, no list reads). */
saf3r_status saf3r_dense_attn(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const void *v_dev,
                              const saf3r_shape *shape, void *out_dev, int out_is_fp32, float *lse_dev_or_null,
                              void *cuda_stream);

/* End-to-end convenience for HOST buffers (one global-attention layer): copies q/k/v (contiguous [H][N][D] bf16, ideally
 * pinned) to the device scratch, runs select + sparse_attn, copies the bf16 output back to out_host; returns after
 * enqueueing (synchronise `cuda_stream` before reading out_host).  The work is pipelined over up to nine groups of heads (the last one a single head, to keep the exposed tail short)
 * on context-owned side streams that are forked from and joined back to `cuda_stream` with events, so that the copies of
 * one group overlap the compute of another; to `cuda_stream` it behaves like one ordered operation.
 * scratch_dev must hold saf3r_layer_host_scratch_bytes(...) bytes; shape strides are ignored (contiguous). */
saf3r_status saf3r_layer_host_scratch_bytes(const saf3r_shape *shape, const saf3r_head_cfg *cfg_host, size_t *bytes);
saf3r_status saf3r_layer_host(saf3r_ctx *ctx, const void *q_host, const void *k_host, const void *v_host,
                              const saf3r_shape *shape, const saf3r_head_cfg *cfg_host, void *scratch_dev,
                              size_t scratch_bytes, void *out_host, void *cuda_stream);

/* Launch plan of saf3r_select for (shape, cfg) on this context's device (host only; a testing aid): *strip_rows = q-block rows
 * scored per CTA of the score + select kernel (0 when no head is BLOCK_TOPK), *smem_bytes = its dynamic shared memory.  A closed
 * form of (shape, cfg, SM count); SAF3R_ERR_UNSUPPORTED when NB is too large for the kernel (the same answer saf3r_select gives,
 * before it enqueues anything).  Either output pointer may be NULL. */
saf3r_status saf3r_select_plan(const saf3r_ctx *ctx, const saf3r_shape *shape, const saf3r_head_cfg *cfg_host, int32_t *strip_rows,
                               size_t *smem_bytes);

/* Number of kernels the library has launched on this context since creation (for bench.py's gpu_launches). */
int64_t saf3r_launch_count(const saf3r_ctx *ctx);

/* ---- Token-granular variants: the paper's own token-level definitions ---------------------------------
 * All of them run the dense mode of the attention kernel over a key/value token set that differs from the query's.
 *
 * saf3r_token_stride_attn: Uniform Sampling Kernel at token level, "selects key positions with a fixed stride"
 *   (s = 32, 64 in Tab. 6/7, L241): every query attends the key tokens {offset + i*stride < N}.  No gather: K and
 *   V are read through a strided TMA view.  stride >= 1, 0 <= offset < min(stride, N).  One launch.
 * saf3r_token_probe_select: Query-Probe Top-K at token level: qbar = (1/N) sum_i q_i,
 *   p[j] = qbar . k_j / sqrt(D) for every key token j, the K tokens with the largest p (score desc, index asc) written
 *   ascending to idx_dev[h][0..K) (int32, [H][K]).  1 <= K <= N, the same K for every head of the call.  Three launches.
 * saf3r_token_set_attn: every query of head h attends the key tokens idx_dev[h][0..K) (ascending, unique, < N; the output of
 *   saf3r_token_probe_select or any caller-made set): gathers those K/V rows into the workspace and runs the dense mode over
 *   them.  Two launches.
 * saf3r_token_query_sizes: workspace bytes of the two calls above (host only). */
saf3r_status saf3r_token_stride_attn(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const void *v_dev,
                                     const saf3r_shape *shape, int32_t stride, int32_t offset, void *out_dev, int out_is_fp32,
                                     float *lse_dev_or_null, void *cuda_stream);
saf3r_status saf3r_token_query_sizes(const saf3r_shape *shape, int32_t K, size_t *select_workspace_bytes,
                                     size_t *attn_workspace_bytes);
saf3r_status saf3r_token_probe_select(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const saf3r_shape *shape, int32_t K,
                                      void *workspace_dev, size_t workspace_bytes, int32_t *idx_dev, void *cuda_stream);
saf3r_status saf3r_token_set_attn(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const void *v_dev,
                                  const saf3r_shape *shape, const int32_t *idx_dev, int32_t K, void *workspace_dev,
                                  size_t workspace_bytes, void *out_dev, int out_is_fp32, float *lse_dev_or_null,
                                  void *cuda_stream);

/* ---- saf3r_token_probe_select for callers that must not allocate device memory -------------------------------------------
 * Who this is for.  Some hosts of this library cannot obtain device memory at the moment they need a result: a plug-in inside
 * an inference server or engine whose memory planner has already claimed the GPU and hands the plug-in only its input and
 * output buffers; a process held under a fixed device-memory quota; a latency-critical loop that may not take the device-wide
 * stall a cudaMalloc / cudaFree implies.  For them every other selection call is unusable, because saf3r_create allocates
 * (a counter and the key-norm ring) and saf3r_token_probe_select wants a caller-made workspace.
 *
 * What it is.  The same three launches as saf3r_token_probe_select (Query-Probe Top-K at token level, PAPER.md:L98, L122-124:
 * qbar = (1/N) sum_i q_i, p[j] = qbar . k_j / sqrt(D), the K key tokens with the largest p written ascending to idx_dev[h][0..K)),
 * the same kernels, hence the same idx bit for bit - but it takes no context and no workspace.  Its scratch (partial query
 * sums, one 32-bit key per (head, token), one histogram per head) lives in a fixed array compiled into the library,
 * SAF3R_NOALLOC_SCRATCH_BYTES (about 4.6 MiB) of device memory that every GPU which loads libsaf3r.so holds from module load
 * until the process exits, whether or not this call is ever made.
 *
 * Limit.  num_heads * N <= SAF3R_NOALLOC_MAX_KEYS (2^20; e.g. 16 heads x 32 frames x 1374 tokens = 703 488 fits, the 100-frame
 * configuration does not).  Anything larger is refused with SAF3R_ERR_CAPACITY before a kernel is enqueued; use
 * saf3r_token_probe_select with your own workspace then.  The other argument rules are those of saf3r_token_probe_select.
 *
 * Device and first call.  It works on the CURRENT CUDA device of the calling thread (there is no context to name one); q, k and
 * idx must live there, and the device must be sm_100 (SAF3R_ERR_UNSUPPORTED otherwise).  The first call on each device looks up
 * the device address of the built-in array (cudaGetSymbolAddress, which may make the runtime load the library's code onto that
 * device) and remembers it; later calls only launch.  Make that first call during start-up, before any stream capture begins.
 * It calls no cudaMalloc / cudaFree / cudaMallocAsync and no library routine that allocates.
 *
 * Sharing.  There is ONE array per device and every call uses it.  It keeps whatever the previous call left; the call itself
 * re-zeroes the part that has to start at zero (the histograms, by its first kernel), so nothing needs clearing between calls.
 * Two calls of one process whose kernels can run at the same time on one device (different streams, or different host threads)
 * overwrite each other's scratch and return garbage without any error: keep all calls on a device in one stream order, or order
 * them with events.  Separate processes each have their own copy and do not interfere.
 *
 * Errors.  Returns a saf3r_status; when err_buf != NULL and err_len > 0 a NUL-terminated message is written there on failure
 * (there is no context to hold it).  Enqueues on cuda_stream and returns; thread-safe on the host side. */
#define SAF3R_NOALLOC_MAX_KEYS (1 << 20)
#define SAF3R_NOALLOC_SCRATCH_BYTES (147456 + 4 * SAF3R_NOALLOC_MAX_KEYS + 8192 * SAF3R_MAX_HEADS)
saf3r_status saf3r_token_probe_select_noalloc(const void *q_dev, const void *k_dev, const saf3r_shape *shape, int32_t K,
                                              int32_t *idx_dev, void *cuda_stream, char *err_buf, size_t err_len);

/* ---- Token-wise per-frame Top-K: the paper's primary definition of the DINO Top-K kernel (SURVEY 8(f) NEXT-2 iii) ----------------
 * "we pre-compute the cosine similarity between each patch token and all other patch tokens using the DINO features, and select
 * the Top-K most similar tokens from each frame as the keys and values for attention"; the indices are computed
 * once per sequence, "cached and reused by all subsequent DINO Top-K kernels" (L126); K = 16..128 per frame (L161), K = 2 / 4
 * attend 0.2 % / 0.4 % of the keys (L242, L249).  Reading A19: every token of every frame is a candidate, the query's
 * own frame and the query itself included.
 *
 * saf3r_token_topk_select: features feat_dev [N][64] bf16 (per sequence, shared by heads and layers; shape->stride_token is the
 *   row stride, num_heads / stride_head / block are ignored) -> idx_dev int32 [N][S][K]: for query token i and frame g the K tokens
 *   of frame g with the largest cosine similarity (score desc, index asc), ascending.  The N x N similarity runs on the tensor
 *   cores a strip of query tiles at a time (strip keys in the workspace); 1 + 2 * ceil(NB128 / strips) launches.
 * saf3r_token_lists_count / _fill: turn idx into what the attention kernel consumes, per q-tile of `block` queries: the union of
 *   its queries' keys, packed over the frames into tiles of `block` gathered key tokens (key_idx, -1 = padding), and one bit per
 *   (query row, key column) of every tile (mask: [tile][block][block/32] uint32).  Tile counts depend on the data: _count writes
 *   tile_ptr_dev[0 .. NB] (offsets; tile_ptr_dev[NB] = total tiles), the caller sizes key_idx (total * block int32) and mask from it
 *   (or from the worst case *max_tiles of saf3r_token_topk_query_sizes) and calls _fill with the same tile_ptr.  A q-tile that does
 *   not fit capacity_tiles is left unwritten.  Both depend only on idx: once per sequence, shared by all heads and layers.
 * saf3r_token_lists_attn: o_i = sum_j softmax_j(q_i.k_j/sqrt(D)) v_j over the keys j of query i's own list: the block-sparse kernel
 *   with K/V rows gathered by index (cp.async) and the bit mask applied before the row max; q, k, v, out, lse as in
 *   saf3r_sparse_attn; the lists are shared by all heads of the call.  Requires tile_ptr[NB] <= capacity_tiles (tile_ptr lives on
 *   the device, so the call cannot check it on the host): a q-tile whose tile range ends beyond capacity_tiles - what a _fill with
 *   too small a capacity leaves unwritten - is skipped on the device, its rows come out zero with lse = -inf, and nothing is read
 *   outside key_idx / mask.  key_idx entries outside [0, N) are treated as padding, never dereferenced. */
typedef struct {
  int64_t *tile_ptr;       /* dev, [NB + 1]: tiles of q-tile I = [tile_ptr[I], tile_ptr[I+1]) */
  int32_t *key_idx;        /* dev, [capacity_tiles * block]: gathered key token of every tile column, -1 = padding */
  uint32_t *mask;          /* dev, [capacity_tiles][block][block/32]: bit c of row r = query r of the q-tile keeps column c */
  int64_t capacity_tiles;
} saf3r_token_lists;
saf3r_status saf3r_token_topk_query_sizes(const saf3r_shape *shape, int32_t K, size_t *select_workspace_bytes, int64_t *idx_entries,
                                          int64_t *max_tiles);
saf3r_status saf3r_token_topk_select(saf3r_ctx *ctx, const void *feat_dev, const saf3r_shape *shape, int32_t K, void *workspace_dev,
                                     size_t workspace_bytes, int32_t *idx_dev, void *cuda_stream);
saf3r_status saf3r_token_lists_count(saf3r_ctx *ctx, const saf3r_shape *shape, int32_t K, const int32_t *idx_dev,
                                     int64_t *tile_ptr_dev, void *cuda_stream);
saf3r_status saf3r_token_lists_fill(saf3r_ctx *ctx, const saf3r_shape *shape, int32_t K, const int32_t *idx_dev,
                                    const saf3r_token_lists *lists, void *cuda_stream);
saf3r_status saf3r_token_lists_attn(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const void *v_dev,
                                    const saf3r_shape *shape, const saf3r_token_lists *lists, void *out_dev, int out_is_fp32,
                                    float *lse_dev_or_null, void *cuda_stream);

/* ---- Static kernel, "broadcast the first frame's local attention map" -----------------
 * Reading (A18): the attention of a position head is content-independent and "fixed across all image blocks", so
 * every T x T image block (f, g) of the N x N map is frame 0's local map P0 = softmax(Q0 K0^T / sqrt(D)) (rows normalised over
 * the whole row: P0 / S).  Hence, for every frame f and in-frame position p,
 *     o[f*T + p] = sum_p' P0[p][p'] * vbar[p'],   vbar[p'] = (1/S) sum_g v[g*T + p'],
 * and lse[f*T + p] = ln sum_p' exp(q[p] . k[p'] / sqrt(D)) + ln S.  Cost O(T^2 D + N D) per head instead of O(N^2 D): logits are
 * computed for frame 0 only and re-used for every frame pair.  Applies to ALL heads of the call (fold the position heads of a
 * layer into one call through the strides).  q, k, v, out, lse as in saf3r_dense_attn; workspace_dev: device scratch of
 * saf3r_static_broadcast_workspace_bytes(shape) bytes, 16-byte aligned (K0 copy, vbar in bf16, frame 0's lse).  Three launches
 * (+ the key-norm pass of the attention kernel); enqueues and returns. */
saf3r_status saf3r_static_broadcast_workspace_bytes(const saf3r_shape *shape, size_t *bytes);
saf3r_status saf3r_static_broadcast_attn(saf3r_ctx *ctx, const void *q_dev, const void *k_dev, const void *v_dev,
                                         const saf3r_shape *shape, void *workspace_dev, size_t workspace_bytes, void *out_dev,
                                         int out_is_fp32, float *lse_dev_or_null, void *cuda_stream);

/* ---- Offline head profiling aid (Eq. 1) ------------------------------------------------
 * E(c) = E_calib[ ||O_full - O_sparse||^2 / ||O_full||^2 ] per head.  saf3r_nmse_accumulate ADDS, for every head h of the call,
 * sum (o_full - o_sparse)^2 to num_den_dev[h] and sum o_full^2 to num_den_dev[H + h] (double accumulators, caller-zeroed, so that
 * several calibration samples can be accumulated); the caller divides.  o_full / o_sparse: two attention outputs with the
 * layout of `shape` (both bf16 or both fp32).  One launch; enqueues and returns. */
saf3r_status saf3r_nmse_accumulate(saf3r_ctx *ctx, const void *o_full_dev, const void *o_sparse_dev, const saf3r_shape *shape,
                                   int is_fp32, double *num_den_dev, void *cuda_stream);

/* Measurement aid ("select ms split into pool and score+select stages").  When enabled, saf3r_select records
 * CUDA events on its stream before the pool launch, between the two launches and after the select launch (three
 * cudaEventRecord calls, no synchronisation).  saf3r_last_select_stage_ms blocks until the last timed saf3r_select has
 * finished and returns the two stage durations in milliseconds: pool_ms = the first launch (pooling, row_ptr, the lists of the
 * constant-length closed-form heads), select_ms = the second launch (the probe of QUERY_PROBE heads, block scores, top-n, every
 * other list). */
saf3r_status saf3r_set_stage_timing(saf3r_ctx *ctx, int enable);
saf3r_status saf3r_last_select_stage_ms(saf3r_ctx *ctx, float *pool_ms, float *select_ms);

#ifdef __cplusplus
}
#endif
#endif /* SAF3R_H_ */
