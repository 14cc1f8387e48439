// C ABI of the SAF3R hot path (include/saf3r.h): argument validation, host-side list sizing, tensor maps, launches.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <string>
#include <vector>

#include "saf3r.h"
#include "attn_kernel.cuh"
#include "select_kernels.cuh"
#include "token_kernels.cuh"
#include "tokenwise_kernels.cuh"

using namespace saf3r;

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct MapKey {
  const void *ptr;
  int64_t N, stride_head, stride_token;
  int32_t H, B;
  bool operator==(const MapKey &o) const {
    return ptr == o.ptr && N == o.N && stride_head == o.stride_head && stride_token == o.stride_token && H == o.H && B == o.B;
  }
};

constexpr size_t kMapCacheEntries = 512;
constexpr uint32_t kKmaxSlots = 256;
constexpr size_t kKmaxSlotFloats = SAF3R_MAX_HEADS + SAF3R_MAX_HEADS / 4;  // kmax[H] floats + head_order[H] bytes

struct saf3r_ctx {
  int device = 0;
  int sm_count = 0;
  EncodeTiledFn encode = nullptr;
  std::string err;
  bool sticky_cuda = false;
  int64_t launches = 0;
  cudaStream_t side[3] = {nullptr, nullptr, nullptr};  // saf3r_layer_host: head-group pipeline (created on first use)
  cudaEvent_t ev_fork = nullptr, ev_join[3] = {nullptr, nullptr, nullptr};
  unsigned long long *counter_dev = nullptr;  // tiny device scratch (saf3r_check_lists)
  // per-head max key norm of the attention calls (knorm_kernel -> saf3r_attn_kernel): a ring of slots, one per call, so that
  // calls in flight on different streams never share one (a slot is reused kKmaxSlots calls later)
  float *kmax_ring = nullptr;
  uint32_t kmax_next = 0;
  bool stage_timing = false;
  cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};  // select: start, after the pool launch, after the select launch
  bool ev_valid = false;
  std::vector<std::pair<MapKey, CUtensorMap>> maps;  // LRU cache, most recently used last (a 24-layer stack holds 72 q/k/v keys)
  struct SizeMemo { int32_t H, S, T, B; saf3r_head_cfg cfg[SAF3R_MAX_HEADS]; int64_t len[SAF3R_MAX_HEADS]; int64_t total; };
  std::vector<SizeMemo> sizes;
};

static saf3r_status fail(saf3r_ctx *ctx, saf3r_status st, const std::string &msg) {
  if (ctx) ctx->err = msg;
  return st;
}
static saf3r_status cuda_fail(saf3r_ctx *ctx, cudaError_t e, const char *where) {
  ctx->sticky_cuda = true;
  ctx->err = std::string(where) + ": " + cudaGetErrorString(e);
  return SAF3R_ERR_CUDA;
}
#define CU_CHECK(call)                                          \
  do {                                                          \
    cudaError_t e__ = (call);                                   \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call); \
  } while (0)

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static const char *validate_shape(const saf3r_shape *s, bool need_strides) {
  if (!s) return "shape is null";
  if (s->num_frames < 1 || s->tokens_per_frame < 1 || s->num_heads < 1) return "num_frames, tokens_per_frame, num_heads must be >= 1";
  if (need_strides) {
    if (s->stride_token < s->head_dim || s->stride_token % 8 || s->stride_head % 8) return "strides must be multiples of 8 elements and stride_token >= head_dim";
  }
  return nullptr;
}
static const char *unsupported_shape(const saf3r_shape *s) {
  if (s->head_dim != 64) return "head_dim must be 64";
  if (s->block != 64 && s->block != 128) return "block must be 64 or 128";
  if (s->num_heads > SAF3R_MAX_HEADS) return "num_heads exceeds SAF3R_MAX_HEADS";
  if ((int64_t)s->num_frames * s->tokens_per_frame > 0x7FFFFFFFll - 256) return "N too large";
  return nullptr;
}
static SelGeom make_geom(const saf3r_shape *s) {
  SelGeom g;
  g.S = s->num_frames; g.T = s->tokens_per_frame; g.H = s->num_heads; g.B = s->block;
  g.N = (int64_t)s->num_frames * s->tokens_per_frame;
  g.NB = (int32_t)((g.N + g.B - 1) / g.B);
  g.stride_head = s->stride_head; g.stride_token = s->stride_token;
  return g;
}
static const char *validate_cfg(const SelGeom &g, const saf3r_head_cfg *cfg, int cache_heads = 0) {
  if (!cfg) return "cfg is null";
  for (int h = 0; h < g.H; ++h) {
    const saf3r_head_cfg &c = cfg[h];
    switch (c.type) {
      case SAF3R_HEAD_CACHED:
        if (cache_heads <= 0) return "CACHED head outside saf3r_select_cached / saf3r_query_sizes, or without a cache";
        if (c.offset < 0 || c.offset >= cache_heads) return "CACHED: offset must name a head of the cache";
        if (c.topk_scope == SAF3R_SCOPE_GLOBAL) {
          if (c.keep_blocks < 1 || c.keep_blocks > g.NB) return "CACHED/GLOBAL: need 1 <= keep_blocks <= NB";
        } else if (c.topk_scope == SAF3R_SCOPE_PER_FRAME) {
          if (c.topk_per_frame < 1) return "CACHED/PER_FRAME: topk_per_frame must be >= 1";
        } else return "CACHED: bad topk_scope";
        break;
      case SAF3R_HEAD_DENSE: break;
      case SAF3R_HEAD_UNIFORM_STRIDE:
        if (c.stride < 0) return "UNIFORM_STRIDE: stride must be >= 0";
        if (c.stride >= 1 && (c.offset < 0 || c.offset >= c.stride || c.offset >= g.NB)) return "UNIFORM_STRIDE: need 0 <= offset < min(stride, NB)";
        if (c.stride == 0 && (c.keep_blocks < 1 || c.keep_blocks > g.NB)) return "UNIFORM_STRIDE: need 1 <= keep_blocks <= NB";
        break;
      case SAF3R_HEAD_STATIC:
        if (c.static_mode < 0 || c.static_mode > 2) return "STATIC: bad static_mode";
        if (c.static_mode == SAF3R_STATIC_ANCHOR && (c.anchor_frame < 0 || c.anchor_frame >= g.S)) return "STATIC/ANCHOR: anchor_frame out of range";
        if (c.static_mode == SAF3R_STATIC_POSITION_BAND && c.band_radius < 0) return "STATIC/POSITION_BAND: band_radius must be >= 0";
        break;
      case SAF3R_HEAD_QUERY_PROBE_TOPK:
        if (c.keep_blocks < 1 || c.keep_blocks > g.NB) return "QUERY_PROBE_TOPK: need 1 <= keep_blocks <= NB";
        break;
      case SAF3R_HEAD_BLOCK_TOPK:
        if (c.score_mode < 0 || c.score_mode > 1) return "BLOCK_TOPK: bad score_mode";
        if (c.topk_scope == SAF3R_SCOPE_GLOBAL) {
          if (c.keep_blocks < 1 || c.keep_blocks > g.NB) return "BLOCK_TOPK/GLOBAL: need 1 <= keep_blocks <= NB";
        } else if (c.topk_scope == SAF3R_SCOPE_PER_FRAME) {
          if (c.topk_per_frame < 1) return "BLOCK_TOPK/PER_FRAME: topk_per_frame must be >= 1";
        } else return "BLOCK_TOPK: bad topk_scope";
        break;
      default: return "unknown head type";
    }
  }
  return nullptr;
}

struct WsLayout {
  size_t qt, kt, qpart, probe, pkeys, counters, total;
};
static WsLayout ws_layout(const SelGeom &g) {
  WsLayout w;
  size_t off = 0;
  w.qt = off; off = align256(off + (size_t)g.H * g.NB * 64 * sizeof(float));
  w.kt = off; off = align256(off + (size_t)g.H * kt_stride(g.NB) * 64 * sizeof(float));
  w.qpart = off; off = align256(off + (size_t)g.H * ((g.NB + kPoolBlocksPerTask - 1) / kPoolBlocksPerTask) * 64 * sizeof(float));
  w.probe = off; off = align256(off + (size_t)g.H * g.NB * sizeof(int32_t));
  w.pkeys = off; off = align256(off + (size_t)g.H * g.NB * sizeof(uint32_t));  // probe rows as keys
  w.counters = off; off = align256(off + kSelCounters * sizeof(int));  // ticket counters and per-head flags of the fused kernel
  w.total = off;
  return w;
}
static int64_t total_entries(const SelGeom &g, const saf3r_head_cfg *cfg, int64_t *per_head = nullptr) {
  int64_t tot = 0;
  for (int h = 0; h < g.H; ++h) {
    const saf3r_head_cfg &c = cfg[h];
    const bool per_row = c.type == SAF3R_HEAD_STATIC && c.static_mode != SAF3R_STATIC_ANCHOR;
    int64_t t = 0;
    if (per_row) {
      for (int64_t I = 0; I < g.NB; ++I) t += row_length(g, c, I);
    } else {
      t = row_length(g, c, 0) * g.NB;
    }
    if (per_head) per_head[h] = t;
    tot += t;
  }
  return tot;
}

extern "C" {

saf3r_status saf3r_create(saf3r_ctx **out, int device) {
  if (!out) return SAF3R_ERR_INVALID_ARG;
  *out = nullptr;
  saf3r_ctx *ctx = new saf3r_ctx();
  ctx->device = device;
  cudaDeviceProp prop;
  cudaError_t e = cudaSetDevice(device);
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) {
    fprintf(stderr, "saf3r_create: no usable CUDA device %d (%s); there is no CPU fallback\n", device, cudaGetErrorString(e));
    delete ctx;
    return SAF3R_ERR_UNSUPPORTED;
  }
  if (prop.major != 10) {
    fprintf(stderr, "saf3r_create: device %d is sm_%d%d; this library is sm_100a only\n", device, prop.major, prop.minor);
    delete ctx;
    return SAF3R_ERR_UNSUPPORTED;
  }
  ctx->sm_count = prop.multiProcessorCount;
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
    fprintf(stderr, "saf3r_create: cuTensorMapEncodeTiled not available\n");
    delete ctx;
    return SAF3R_ERR_UNSUPPORTED;
  }
  ctx->encode = (EncodeTiledFn)fn;
  e = cudaFuncSetAttribute(saf3r_attn_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<128>::kTotal);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(saf3r_attn_kernel<64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<64>::kTotal);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(saf3r_attn_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<128>::kTotal);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(saf3r_attn_kernel<64, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem<64>::kTotal);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(select_fused_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(select_fused_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 72 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(token_sim_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSimSmem);
  if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->counter_dev, sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->kmax_ring, sizeof(float) * kKmaxSlots * kKmaxSlotFloats);
  if (e != cudaSuccess) {
    fprintf(stderr, "saf3r_create: cudaFuncSetAttribute / cudaMalloc failed: %s\n", cudaGetErrorString(e));
    delete ctx;
    return SAF3R_ERR_CUDA;
  }
  *out = ctx;
  return SAF3R_OK;
}

void saf3r_destroy(saf3r_ctx *ctx) {
  if (!ctx) return;
  for (auto &e : ctx->ev)
    if (e) cudaEventDestroy(e);
  if (ctx->counter_dev) cudaFree(ctx->counter_dev);
  if (ctx->kmax_ring) cudaFree(ctx->kmax_ring);
  for (auto &sd : ctx->side)
    if (sd) cudaStreamDestroy(sd);
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  for (auto &e : ctx->ev_join)
    if (e) cudaEventDestroy(e);
  delete ctx;
}

const char *saf3r_last_error(const saf3r_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int64_t saf3r_launch_count(const saf3r_ctx *ctx) { return ctx ? ctx->launches : 0; }

saf3r_status saf3r_set_stage_timing(saf3r_ctx *ctx, int enable) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (enable && !ctx->ev[0]) {
    for (auto &e : ctx->ev) CU_CHECK(cudaEventCreate(&e));
  }
  ctx->stage_timing = enable != 0;
  ctx->ev_valid = false;
  return SAF3R_OK;
}

saf3r_status saf3r_last_select_stage_ms(saf3r_ctx *ctx, float *pool_ms, float *select_ms) {
  if (!ctx || !pool_ms || !select_ms) return SAF3R_ERR_INVALID_ARG;
  if (!ctx->ev_valid) return fail(ctx, SAF3R_ERR_INVALID_ARG, "no timed saf3r_select call yet (saf3r_set_stage_timing)");
  CU_CHECK(cudaEventSynchronize(ctx->ev[2]));
  CU_CHECK(cudaEventElapsedTime(pool_ms, ctx->ev[0], ctx->ev[1]));
  CU_CHECK(cudaEventElapsedTime(select_ms, ctx->ev[1], ctx->ev[2]));
  return SAF3R_OK;
}

saf3r_status saf3r_query_sizes(const saf3r_shape *shape, const saf3r_head_cfg *cfg, int64_t *list_entries, size_t *workspace_bytes) {
  if (validate_shape(shape, false) || !cfg) return SAF3R_ERR_INVALID_ARG;
  if (unsupported_shape(shape)) return SAF3R_ERR_UNSUPPORTED;
  const SelGeom g = make_geom(shape);
  if (validate_cfg(g, cfg, SAF3R_MAX_HEADS)) return SAF3R_ERR_INVALID_ARG;  // CACHED heads: lengths are closed forms too
  if (list_entries) *list_entries = total_entries(g, cfg);
  if (workspace_bytes) *workspace_bytes = ws_layout(g).total;
  return SAF3R_OK;
}

}  // extern "C"


// Launch plan of the score + select kernel: rows per score strip R (16; fewer when R*NB keys do not fit the shared-memory budget of
// two CTAs per SM - then of one - or when the BLOCK_TOPK heads are few, so that the strips cover every SM twice) and the dynamic
// shared memory.  A closed form of (shape, cfg, SM count), computed BEFORE anything is enqueued.
struct SelPlan { int R; size_t smem; const char *unsupported; bool tail_stage; };
static SelPlan select_plan(const SelGeom &g, int n_block, int n_probe, int sm_count) {
  SelPlan p{kSelRows, 0, nullptr, false};
  const size_t row = (size_t)kt_stride(g.NB) * 4;
  if (n_block > 0) {
    const size_t qbytes = 64 * kSelRows * 4;
    size_t budget = 108 * 1024 - qbytes;  // two CTAs per SM
    if (row > budget) budget = 220 * 1024 - qbytes;
    if (row > budget) { p.unsupported = "NB too large for the select kernel"; return p; }
    while ((size_t)p.R * row > budget) --p.R;
    while (p.R > 8 && ((int64_t)n_block * ((g.NB + p.R - 1) / p.R) < 2 * (int64_t)sm_count || g.NB <= 1152)) p.R = (p.R + 1) / 2;  // NB <= 1152: 8-row strips, three CTAs per SM
    p.smem = (size_t)p.R * row + qbytes;
    // staging of the columns left over after the groups of 1024 (score_rows), when they are few
    const int64_t tail_cols = kt_stride(g.NB) - (g.NB / 1024) * 1024;
    p.tail_stage = g.NB >= 1024 && tail_cols <= kSelTailCols && p.smem + 64 * tail_cols * 4 <= (p.smem <= 108 * 1024 ? 108 * 1024 : 220 * 1024);
    if (p.tail_stage) p.smem += 64 * tail_cols * 4;
  }
  if (n_probe > 0) {
    if (row > 220 * 1024) { p.unsupported = "NB too large for the probe stage"; return p; }
    if (p.smem < row) p.smem = row;
    if (p.smem < (size_t)kSelScratch) p.smem = kSelScratch;
  }
  if (p.smem < 4096) p.smem = 4096;  // scratch of the pool / row_ptr tasks
  return p;
}

static saf3r_status select_impl(saf3r_ctx *ctx, const void *q, const void *k, const saf3r_shape *shape, const saf3r_head_cfg *cfg,
                                const saf3r_lists *cache, int cache_heads, void *ws, size_t ws_bytes, saf3r_lists *lists,
                                void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  const SelGeom g = make_geom(shape);
  if (cache && (!cache->row_ptr || !cache->col_idx || cache_heads < 1 || cache_heads > SAF3R_MAX_HEADS))
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "cache has null arrays or a bad head count");
  if (const char *m = validate_cfg(g, cfg, cache ? cache_heads : 0)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (!q || !k || !ws || !lists || !lists->row_ptr || !lists->col_idx) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)q | (uintptr_t)k) & 15) return fail(ctx, SAF3R_ERR_INVALID_ARG, "q/k must be 16-byte aligned");
  const WsLayout w = ws_layout(g);
  struct { int64_t len[SAF3R_MAX_HEADS]; } hint;  // per-head list totals (closed forms)
  memset(&hint, 0, sizeof hint);
  // list sizes are a closed form of (shape, cfg); the per-row-length STATIC rules cost O(NB) .. O(NB*S) host work, so the last
  // few (shape, cfg) -> sizes results are memoised
  int64_t need = -1;
  for (auto &e : ctx->sizes)
    if (e.H == g.H && e.S == g.S && e.T == g.T && e.B == g.B && memcmp(e.cfg, cfg, sizeof(saf3r_head_cfg) * g.H) == 0) {
      memcpy(hint.len, e.len, sizeof hint.len);
      need = e.total;
    }
  if (need < 0) {
    need = total_entries(g, cfg, hint.len);
    saf3r_ctx::SizeMemo m;
    m.H = g.H; m.S = g.S; m.T = g.T; m.B = g.B; m.total = need;
    memset(m.cfg, 0, sizeof m.cfg);
    memcpy(m.cfg, cfg, sizeof(saf3r_head_cfg) * g.H);
    memcpy(m.len, hint.len, sizeof m.len);
    if (ctx->sizes.size() >= 64) ctx->sizes.erase(ctx->sizes.begin());
    ctx->sizes.push_back(m);
  }
  if (ws_bytes < w.total || lists->capacity < need) {
    char buf[160];
    snprintf(buf, sizeof buf, "capacity: need %lld list entries (have %lld), %zu workspace bytes (have %zu)", (long long)need,
             (long long)lists->capacity, w.total, ws_bytes);
    return fail(ctx, SAF3R_ERR_CAPACITY, buf);
  }
  cudaStream_t st = (cudaStream_t)stream_;
  uint8_t *wsb = (uint8_t *)ws;
  float *qt = (float *)(wsb + w.qt), *kt = (float *)(wsb + w.kt) , *qpart = (float *)(wsb + w.qpart);
  int32_t *probe = (int32_t *)(wsb + w.probe);

  HeadCfgArray ca;
  memset(&ca, 0, sizeof ca);
  PoolJobs jobs;
  memset(&jobs, 0, sizeof jobs);
  RowPtrPlan plan;
  memset(&plan, 0, sizeof plan);
  HeadSets sets;
  memset(&sets, 0, sizeof sets);
  int64_t base = 0;
  for (int h = 0; h < g.H; ++h) {
    ca.c[h] = cfg[h];
    const bool per_row = cfg[h].type == SAF3R_HEAD_STATIC && cfg[h].static_mode != SAF3R_STATIC_ANCHOR;
    if (cfg[h].type == SAF3R_HEAD_CACHED) sets.cached[sets.n_cached++] = (uint8_t)h;
    else if (cfg[h].type == SAF3R_HEAD_BLOCK_TOPK) sets.block[sets.n_block++] = (uint8_t)h;
    else if (cfg[h].type == SAF3R_HEAD_QUERY_PROBE_TOPK) sets.probe[sets.n_probe++] = (uint8_t)h;
    else if (per_row) sets.light[sets.n_light++] = (uint8_t)h;
    else sets.emit[sets.n_emit++] = (uint8_t)h;
    plan.const_len[h] = per_row ? -1 : (int32_t)row_length(g, cfg[h], 0);
    plan.head_base[h] = base;
    base += hint.len[h];
  }
  plan.head_base[g.H] = base;
  // pool jobs: BLOCK_TOPK heads first (their score strips then run under the pooling of the QUERY_PROBE heads)
  for (int pass = 0; pass < 2; ++pass)
    for (int h = 0; h < g.H; ++h) {
      const bool probe = cfg[h].type == SAF3R_HEAD_QUERY_PROBE_TOPK, block = cfg[h].type == SAF3R_HEAD_BLOCK_TOPK;
      if (!(pass == 0 ? block : probe)) continue;
      for (int which = 0; which < 2; ++which) {
        jobs.head[jobs.n] = (uint8_t)h;
        jobs.which[jobs.n] = (uint8_t)which;
        jobs.cosine[jobs.n] = (uint8_t)(block && cfg[h].score_mode == SAF3R_SCORE_COSINE);
        jobs.probe[jobs.n] = (uint8_t)probe;
        ++jobs.n;
      }
    }
  // the launch plan first: an UNSUPPORTED shape must be reported before anything is enqueued (saf3r.h "Asynchrony")
  const SelPlan sp = select_plan(g, sets.n_block, sets.n_probe, ctx->sm_count);
  if (sp.unsupported) return fail(ctx, SAF3R_ERR_UNSUPPORTED, sp.unsupported);
  const int tasks_per_job = (g.NB + kPoolBlocksPerTask - 1) / kPoolBlocksPerTask;
  const int light_chunks = (g.NB + kLightRows - 1) / kLightRows;
  FusedPlan fp;
  memset(&fp, 0, sizeof fp);
  fp.R = sp.R;
  fp.tail_stage = sp.tail_stage ? 1 : 0;
  fp.strips = (g.NB + sp.R - 1) / sp.R;
  fp.light_chunks = light_chunks;
  fp.pool_need = 2 * tasks_per_job;
  fp.n_rowptr = g.H;
  fp.n_pool_a = 2 * sets.n_block * tasks_per_job;   // jobs are ordered BLOCK_TOPK heads first (see above)
  fp.n_pool_b = 2 * sets.n_probe * tasks_per_job;
  fp.n_x = sets.n_block * fp.strips;                // score strips: mixed into the pooling of the QUERY_PROBE heads
  fp.pchunks = (g.NB + kProbeChunk - 1) / kProbeChunk;
  fp.n_pscore = sets.n_probe * fp.pchunks;          // everything from here on follows ALL pool tasks
  fp.n_probe = sets.n_probe;
  fp.n_light = (sets.n_light + sets.n_cached) * light_chunks;
  fp.n_emit = sets.n_emit * light_chunks;
  fp.n_rep = sets.n_probe * light_chunks;
  fp.period = fp.n_x > 0 && fp.n_pool_b / fp.n_x > 1 ? fp.n_pool_b / fp.n_x : 1;
  const int n_tasks = fp.n_rowptr + fp.n_pool_a + fp.n_pool_b + fp.n_x + fp.n_pscore + fp.n_probe + fp.n_light + fp.n_emit + fp.n_rep;
  int *counters = (int *)(wsb + w.counters);
  CU_CHECK(cudaMemsetAsync(counters, 0, kSelCounters * sizeof(int), st));
  auto launch = [&](int t_begin, int t_end, int counter) {
    fp.t_begin = t_begin; fp.t_end = t_end; fp.counter = counter;
    // three CTAs per SM when the strips are short and the rows fit the 36-keys-per-lane register top-n (80 registers per thread):
    // a CTA that is busy with a latency-bound score strip then leaves two CTAs of the SM streaming Q / K
    const bool occ3 = sp.R <= 8 && g.NB <= 1152 && sp.smem <= 72 * 1024;
    const int per_sm = occ3 ? 3 : 2;
    const int ctas = t_end - t_begin < per_sm * ctx->sm_count ? t_end - t_begin : per_sm * ctx->sm_count;
    if (ctas <= 0) return;
    (occ3 ? select_fused_kernel<3> : select_fused_kernel<2>)<<<ctas, 256, sp.smem, st>>>((const __nv_bfloat16 *)q, (const __nv_bfloat16 *)k, qt, kt, qpart, (uint32_t *)(wsb + w.pkeys), probe, lists->row_ptr,
                                                   lists->col_idx, (const int64_t *)(cache ? cache->row_ptr : nullptr),
                                                   (const int32_t *)(cache ? cache->col_idx : nullptr), counters, g, jobs, plan, ca, sets, fp);
    ctx->launches += 1;
  };
  if (!ctx->stage_timing) {
    launch(0, n_tasks, 0);   // ONE launch: the dependent tasks run under the pooling of the QUERY_PROBE heads
  } else {
    // measurement aid: the same kernel as two launches, pooling (+ row_ptr) first, everything else second, with events around them
    fp.period = fp.n_pool_b + 1;  // no mixing: all pool tasks come before the first dependent task
    const int n_first = fp.n_rowptr + fp.n_pool_a + fp.n_pool_b;
    cudaEventRecord(ctx->ev[0], st);
    launch(0, n_first, 0);
    cudaEventRecord(ctx->ev[1], st);
    launch(n_first, n_tasks, 1);
    cudaEventRecord(ctx->ev[2], st);
    ctx->ev_valid = true;
  }
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

extern "C" {

saf3r_status saf3r_select(saf3r_ctx *ctx, const void *q, const void *k, const saf3r_shape *shape, const saf3r_head_cfg *cfg,
                          void *ws, size_t ws_bytes, saf3r_lists *lists, void *stream) {
  return select_impl(ctx, q, k, shape, cfg, nullptr, 0, ws, ws_bytes, lists, stream);
}

saf3r_status saf3r_select_cached(saf3r_ctx *ctx, const void *q, const void *k, const saf3r_shape *shape, const saf3r_head_cfg *cfg,
                                 const saf3r_lists *cache, int32_t cache_heads, void *ws, size_t ws_bytes, saf3r_lists *lists,
                                 void *stream) {
  return select_impl(ctx, q, k, shape, cfg, cache, cache ? cache_heads : 0, ws, ws_bytes, lists, stream);
}

}  // extern "C"

static saf3r_status get_map(saf3r_ctx *ctx, const void *ptr, const SelGeom &g, CUtensorMap *out) {
  MapKey key{ptr, g.N, g.stride_head, g.stride_token, g.H, g.B};
  for (size_t i = ctx->maps.size(); i-- > 0;)  // most recently used at the back
    if (ctx->maps[i].first == key) {
      *out = ctx->maps[i].second;
      if (i + 1 != ctx->maps.size()) {  // LRU: move the hit to the back
        auto hit = ctx->maps[i];
        ctx->maps.erase(ctx->maps.begin() + (long)i);
        ctx->maps.push_back(hit);
      }
      return SAF3R_OK;
    }
  CUtensorMap m;
  const cuuint64_t dims[3] = {64, (cuuint64_t)g.N, (cuuint64_t)g.H};
  const cuuint64_t strides[2] = {(cuuint64_t)g.stride_token * 2, (cuuint64_t)g.stride_head * 2};
  const cuuint32_t box[3] = {64, (cuuint32_t)g.B, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  // with one head the head stride is irrelevant but must still be a valid (multiple of 16, >= row extent) value
  cuuint64_t strides_fixed[2] = {strides[0], strides[1]};
  if (g.H == 1 && strides_fixed[1] < strides_fixed[0] * (cuuint64_t)g.N) strides_fixed[1] = strides_fixed[0] * (cuuint64_t)g.N;
  CUresult r = ctx->encode(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(ptr), dims, strides_fixed, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[96];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return fail(ctx, SAF3R_ERR_INVALID_ARG, buf);
  }
  if (ctx->maps.size() >= kMapCacheEntries) ctx->maps.erase(ctx->maps.begin());  // evict the least recently used
  ctx->maps.emplace_back(key, m);
  *out = m;
  return SAF3R_OK;
}

struct KvGeom {  // key/value token set that differs from the query's (token-granular variants); n == 0: same as q
  int64_t n, stride_head, stride_token;
};

static saf3r_status attn_common(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape,
                                const saf3r_lists *lists, void *out, int out_is_fp32, float *lse, void *stream_,
                                const KvGeom *kv = nullptr) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!q || !k || !v || !out) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out) & 15) return fail(ctx, SAF3R_ERR_INVALID_ARG, "q/k/v/out must be 16-byte aligned");
  if (lists && (!lists->row_ptr || !lists->col_idx)) return fail(ctx, SAF3R_ERR_INVALID_ARG, "lists has null arrays");
  const SelGeom g = make_geom(shape);
  SelGeom gk = g;
  if (kv) {
    if (kv->n < 1 || kv->n > 0x7FFFFFFFll - 256) return fail(ctx, SAF3R_ERR_INVALID_ARG, "n_kv out of range");
    if (kv->stride_token < shape->head_dim || kv->stride_token % 8 || kv->stride_head % 8)
      return fail(ctx, SAF3R_ERR_INVALID_ARG, "kv strides must be multiples of 8 elements and kv_stride_token >= head_dim");
    gk.N = kv->n;
    gk.NB = (int32_t)((kv->n + g.B - 1) / g.B);
    gk.stride_head = kv->stride_head;
    gk.stride_token = kv->stride_token;
  }
  CUtensorMap mq, mk, mv;
  saf3r_status s;
  if ((s = get_map(ctx, q, g, &mq)) != SAF3R_OK) return s;
  if ((s = get_map(ctx, k, gk, &mk)) != SAF3R_OK) return s;
  if ((s = get_map(ctx, v, gk, &mv)) != SAF3R_OK) return s;
  AttnParams p;
  p.row_ptr = lists ? lists->row_ptr : nullptr;
  p.col_idx = lists ? lists->col_idx : nullptr;
  p.out = out;
  p.lse = lse;
  p.out_stride_head = shape->stride_head;
  p.out_stride_token = shape->stride_token;
  p.N = (int32_t)g.N; p.NB = g.NB; p.H = g.H;
  p.N_kv = (int32_t)gk.N; p.NB_kv = gk.NB;
  p.out_fp32 = out_is_fp32 ? 1 : 0;
  p.scale_log2 = (float)(1.4426950408889634 / sqrt((double)shape->head_dim));
  cudaStream_t st = (cudaStream_t)stream_;
  // max key norm per head (one streaming pass over K) for the kernel's frozen-max fast path; worth it from a few k-tiles per
  // q-block on (the pass reads K once, the attention reads it NB times through L2)
  // The same launch orders the heads by list length, longest first (one CTA reads row_ptr; hand-made lists are balanced too).
  p.kmax = nullptr;
  p.head_order = nullptr;
  if (gk.NB >= 4) {
    float *slot = ctx->kmax_ring + (size_t)(ctx->kmax_next++ % kKmaxSlots) * kKmaxSlotFloats;
    CU_CHECK(cudaMemsetAsync(slot, 0, sizeof(float) * g.H, st));
    knorm_kernel<<<dim3((unsigned)((gk.N + kKnormRows - 1) / kKnormRows), g.H), 256, 0, st>>>(
        (const __nv_bfloat16 *)k, gk.N, gk.stride_head, gk.stride_token, slot, p.row_ptr, g.NB, reinterpret_cast<uint8_t *>(slot + SAF3R_MAX_HEADS));
    ctx->launches += 1;
    p.kmax = slot;
    p.head_order = reinterpret_cast<const uint8_t *>(slot + SAF3R_MAX_HEADS);
  }
  dim3 grid(g.NB, g.H);
  p.tile_ptr = nullptr; p.key_idx = nullptr; p.mask = nullptr; p.k_base = p.v_base = nullptr; p.kv_stride_head = p.kv_stride_token = 0;
  if (g.B == 128)
    saf3r_attn_kernel<128, false><<<grid, kAttnThreads, AttnSmem<128>::kTotal, st>>>(mq, mk, mv, p);
  else
    saf3r_attn_kernel<64, false><<<grid, kAttnThreads, AttnSmem<64>::kTotal, st>>>(mq, mk, mv, p);
  ctx->launches += 1;
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

extern "C" {

saf3r_status saf3r_sparse_attn(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape,
                               const saf3r_lists *lists, void *out, int out_is_fp32, float *lse, void *stream) {
  if (!lists) return fail(ctx, SAF3R_ERR_INVALID_ARG, "lists is null");
  return attn_common(ctx, q, k, v, shape, lists, out, out_is_fp32, lse, stream);
}

saf3r_status saf3r_select_plan(const saf3r_ctx *ctx, const saf3r_shape *shape, const saf3r_head_cfg *cfg, int32_t *strip_rows,
                               size_t *smem_bytes) {
  if (!ctx || validate_shape(shape, false) || !cfg) return SAF3R_ERR_INVALID_ARG;
  if (unsupported_shape(shape)) return SAF3R_ERR_UNSUPPORTED;
  const SelGeom g = make_geom(shape);
  if (validate_cfg(g, cfg, SAF3R_MAX_HEADS)) return SAF3R_ERR_INVALID_ARG;
  int nb = 0, np = 0;
  for (int h = 0; h < g.H; ++h) {
    nb += cfg[h].type == SAF3R_HEAD_BLOCK_TOPK;
    np += cfg[h].type == SAF3R_HEAD_QUERY_PROBE_TOPK;
  }
  const SelPlan sp = select_plan(g, nb, np, ctx->sm_count);
  if (sp.unsupported) return SAF3R_ERR_UNSUPPORTED;
  if (strip_rows) *strip_rows = nb > 0 ? sp.R : 0;
  if (smem_bytes) *smem_bytes = sp.smem;
  return SAF3R_OK;
}

saf3r_status saf3r_check_lists(saf3r_ctx *ctx, const saf3r_shape *shape, const saf3r_lists *lists, int64_t *bad_rows, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, false)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!lists || !lists->row_ptr || !lists->col_idx || !bad_rows) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  const SelGeom g = make_geom(shape);
  cudaStream_t st = (cudaStream_t)stream_;
  unsigned long long *bad = ctx->counter_dev, host = 0;  // allocated by saf3r_create
  CU_CHECK(cudaMemsetAsync(bad, 0, sizeof *bad, st));
  const int64_t rows = (int64_t)g.H * g.NB;
  check_lists_kernel<<<(unsigned)((rows + 255) / 256 < 4096 ? (rows + 255) / 256 : 4096), 256, 0, st>>>(lists->row_ptr, lists->col_idx,
                                                                                                       rows, g.NB, lists->capacity, bad);
  ctx->launches += 1;
  CU_CHECK(cudaMemcpyAsync(&host, bad, sizeof host, cudaMemcpyDeviceToHost, st));
  CU_CHECK(cudaStreamSynchronize(st));
  *bad_rows = (int64_t)host;
  return SAF3R_OK;
}

saf3r_status saf3r_union_lists(saf3r_ctx *ctx, const saf3r_shape *shape, const saf3r_lists *a, const saf3r_lists *b, saf3r_lists *out,
                               void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, false)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!a || !b || !out || !a->row_ptr || !a->col_idx || !b->row_ptr || !b->col_idx || !out->row_ptr || !out->col_idx)
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (out->row_ptr == a->row_ptr || out->row_ptr == b->row_ptr || out->col_idx == a->col_idx || out->col_idx == b->col_idx)
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "the union is not computed in place: out must not alias an input");
  const SelGeom g = make_geom(shape);
  const int64_t rows = (int64_t)g.H * g.NB;
  cudaStream_t st = (cudaStream_t)stream_;
  const unsigned ctas = (unsigned)((rows + 127) / 128);
  union_rows_kernel<false><<<ctas, 128, 0, st>>>(a->row_ptr, a->col_idx, b->row_ptr, b->col_idx, out->row_ptr, out->col_idx, rows, out->capacity);
  scan_row_ptr_kernel<<<1, 1024, 0, st>>>(out->row_ptr, rows);
  union_rows_kernel<true><<<ctas, 128, 0, st>>>(a->row_ptr, a->col_idx, b->row_ptr, b->col_idx, out->row_ptr, out->col_idx, rows, out->capacity);
  ctx->launches += 3;
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

saf3r_status saf3r_dense_attn(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape, void *out,
                              int out_is_fp32, float *lse, void *stream) {
  return attn_common(ctx, q, k, v, shape, nullptr, out, out_is_fp32, lse, stream);
}

// ------------------------------------------------------------------------------------------------ token-granular variants
saf3r_status saf3r_token_stride_attn(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape,
                                     int32_t stride, int32_t offset, void *out, int out_is_fp32, float *lse, void *stream) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  const int64_t N = (int64_t)shape->num_frames * shape->tokens_per_frame;
  if (stride < 1 || offset < 0 || offset >= stride || offset >= N)
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "token stride: need stride >= 1 and 0 <= offset < min(stride, N)");
  if (!k || !v) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  const KvGeom kv{(N - offset + stride - 1) / stride, shape->stride_head, shape->stride_token * (int64_t)stride};
  const __nv_bfloat16 *k0 = (const __nv_bfloat16 *)k + (int64_t)offset * shape->stride_token;
  const __nv_bfloat16 *v0 = (const __nv_bfloat16 *)v + (int64_t)offset * shape->stride_token;
  return attn_common(ctx, q, k0, v0, shape, nullptr, out, out_is_fp32, lse, stream, &kv);
}

struct TokWs {
  size_t part, keys, hist1, select_total, kc, vc, attn_total;
  int n_chunks;
};
static TokWs tok_ws(const SelGeom &g, int K) {
  TokWs w;
  w.n_chunks = (int)((g.N + kTokChunk - 1) / kTokChunk);
  size_t off = 0;
  w.part = off; off = align256(off + (size_t)g.H * w.n_chunks * 64 * sizeof(float));
  w.keys = off; off = align256(off + (size_t)g.H * g.N * sizeof(uint32_t));
  w.hist1 = off; off = align256(off + (size_t)g.H * kTokBins1 * sizeof(uint32_t));
  w.select_total = off;
  off = 0;
  w.kc = off; off = align256(off + (size_t)g.H * K * 64 * 2);
  w.vc = off; off = align256(off + (size_t)g.H * K * 64 * 2);
  w.attn_total = off;
  return w;
}

saf3r_status saf3r_token_query_sizes(const saf3r_shape *shape, int32_t K, size_t *select_ws, size_t *attn_ws) {
  if (validate_shape(shape, false)) return SAF3R_ERR_INVALID_ARG;
  if (unsupported_shape(shape)) return SAF3R_ERR_UNSUPPORTED;
  const SelGeom g = make_geom(shape);
  if (K < 1 || K > g.N) return SAF3R_ERR_INVALID_ARG;
  const TokWs w = tok_ws(g, K);
  if (select_ws) *select_ws = w.select_total;
  if (attn_ws) *attn_ws = w.attn_total;
  return SAF3R_OK;
}

saf3r_status saf3r_token_probe_select(saf3r_ctx *ctx, const void *q, const void *k, const saf3r_shape *shape, int32_t K, void *ws,
                                      size_t ws_bytes, int32_t *idx, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  const SelGeom g = make_geom(shape);
  if (K < 1 || K > g.N) return fail(ctx, SAF3R_ERR_INVALID_ARG, "token probe: need 1 <= K <= N");
  if (!q || !k || !ws || !idx) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)q | (uintptr_t)k) & 15) return fail(ctx, SAF3R_ERR_INVALID_ARG, "q/k must be 16-byte aligned");
  const TokWs w = tok_ws(g, K);
  if (ws_bytes < w.select_total) return fail(ctx, SAF3R_ERR_CAPACITY, "workspace too small (saf3r_token_query_sizes)");
  cudaStream_t st = (cudaStream_t)stream_;
  float *part = (float *)((uint8_t *)ws + w.part);
  uint32_t *keys = (uint32_t *)((uint8_t *)ws + w.keys), *hist1 = (uint32_t *)((uint8_t *)ws + w.hist1);
  token_qsum_kernel<<<dim3(w.n_chunks, g.H), 256, 0, st>>>((const __nv_bfloat16 *)q, part, hist1, g);
  token_probe_kernel<<<dim3((unsigned)((g.N + kTokTile - 1) / kTokTile), g.H), 256, 0, st>>>((const __nv_bfloat16 *)k, part, keys, hist1,
                                                                                           g, w.n_chunks);
  token_topk_kernel<<<g.H, 1024, 0, st>>>(keys, hist1, idx, g.N, K);
  ctx->launches += 3;
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ allocation-free token probe
// saf3r_token_probe_select_noalloc (include/saf3r.h): for hosts that cannot get device memory when they call us (a plug-in whose
// engine has planned all of it, a process under a memory quota, a loop that may not stall on cudaMalloc).  The scratch the three
// token-probe kernels need is this array, part of the library image on every device that loads it.  Fixed layout, sized for the
// documented maximum so that it does not depend on the shape of the call:
//   [0, kNaPartBytes)                      partial query sums, H * ceil(N / kTokChunk) * 64 floats (<= 576 rows of 256 B)
//   [kNaPartBytes, +4 * MAX_KEYS)          one order-preserving 32-bit key per (head, key token)
//   [.., + MAX_HEADS * kTokBins1 * 4)      one first-level histogram per head (zeroed by token_qsum_kernel on every call)
constexpr size_t kNaPartBytes = ((size_t)SAF3R_NOALLOC_MAX_KEYS / kTokChunk + SAF3R_MAX_HEADS) * 64 * sizeof(float);
constexpr size_t kNaKeysBytes = (size_t)SAF3R_NOALLOC_MAX_KEYS * sizeof(uint32_t);
constexpr size_t kNaHistBytes = (size_t)SAF3R_MAX_HEADS * kTokBins1 * sizeof(uint32_t);
static_assert(kNaPartBytes % 256 == 0 && kNaKeysBytes % 256 == 0, "sub-buffers of the built-in scratch must stay 256-byte aligned");
static_assert(kNaPartBytes + kNaKeysBytes + kNaHistBytes == (size_t)SAF3R_NOALLOC_SCRATCH_BYTES, "saf3r.h states the size of this array");
static __device__ __align__(256) unsigned char g_noalloc_scratch[SAF3R_NOALLOC_SCRATCH_BYTES];

// In host code `g_noalloc_scratch` is only a handle for the runtime, not an address a kernel can use: the device address differs per
// GPU and has to be asked for with that GPU current.  Looked up once per device and kept; guarded because there is no context
// (and so no single-thread rule) on this path.
constexpr int kNaMaxDevices = 64;
static std::mutex g_noalloc_mu;
static unsigned char *g_noalloc_ptr[kNaMaxDevices] = {};

static saf3r_status noalloc_fail(char *err_buf, size_t err_len, saf3r_status st, const std::string &msg) {
  if (err_buf && err_len) snprintf(err_buf, err_len, "%s", msg.c_str());
  return st;
}

static saf3r_status noalloc_scratch(unsigned char **out, char *err_buf, size_t err_len) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return noalloc_fail(err_buf, err_len, SAF3R_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kNaMaxDevices) return noalloc_fail(err_buf, err_len, SAF3R_ERR_UNSUPPORTED, "device ordinal beyond the per-device table of the built-in scratch");
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {  // first call on this device: the set-up the header asks callers to do before any stream capture
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return noalloc_fail(err_buf, err_len, SAF3R_ERR_CUDA, std::string("cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
    if (major != 10) return noalloc_fail(err_buf, err_len, SAF3R_ERR_UNSUPPORTED, "the current device is not sm_100; this library is sm_100a only and has no CPU fallback");
    unsigned char *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p)
      return noalloc_fail(err_buf, err_len, SAF3R_ERR_CUDA, std::string("cudaGetSymbolAddress(built-in scratch): ") + cudaGetErrorString(e));
    g_noalloc_ptr[dev] = p;
  }
  *out = g_noalloc_ptr[dev];
  return SAF3R_OK;
}

extern "C" {

saf3r_status saf3r_token_probe_select_noalloc(const void *q, const void *k, const saf3r_shape *shape, int32_t K, int32_t *idx,
                                              void *stream_, char *err_buf, size_t err_len) {
  if (err_buf && err_len) err_buf[0] = 0;
  if (const char *m = validate_shape(shape, true)) return noalloc_fail(err_buf, err_len, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return noalloc_fail(err_buf, err_len, SAF3R_ERR_UNSUPPORTED, m);
  const SelGeom g = make_geom(shape);
  if (K < 1 || K > g.N) return noalloc_fail(err_buf, err_len, SAF3R_ERR_INVALID_ARG, "token probe: need 1 <= K <= N");
  if (!q || !k || !idx) return noalloc_fail(err_buf, err_len, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)q | (uintptr_t)k) & 15) return noalloc_fail(err_buf, err_len, SAF3R_ERR_INVALID_ARG, "q/k must be 16-byte aligned");
  if ((int64_t)g.H * g.N > (int64_t)SAF3R_NOALLOC_MAX_KEYS)
    return noalloc_fail(err_buf, err_len, SAF3R_ERR_CAPACITY,
                        "num_heads * N = " + std::to_string((int64_t)g.H * g.N) + " exceeds SAF3R_NOALLOC_MAX_KEYS = " +
                            std::to_string((int64_t)SAF3R_NOALLOC_MAX_KEYS) +
                            ", the size of the built-in scratch: call saf3r_token_probe_select with a workspace of your own");
  const int n_chunks = (int)((g.N + kTokChunk - 1) / kTokChunk);
  if ((size_t)g.H * n_chunks * 64 * sizeof(float) > kNaPartBytes)  // implied by the check above; kept as the layout's own guard
    return noalloc_fail(err_buf, err_len, SAF3R_ERR_CAPACITY, "partial query sums exceed the built-in scratch");
  unsigned char *base = nullptr;
  if (saf3r_status s = noalloc_scratch(&base, err_buf, err_len)) return s;
  cudaStream_t st = (cudaStream_t)stream_;
  float *part = (float *)base;
  uint32_t *keys = (uint32_t *)(base + kNaPartBytes), *hist1 = (uint32_t *)(base + kNaPartBytes + kNaKeysBytes);
  // Same three launches as saf3r_token_probe_select.  Everything read is written earlier in this very call: `part` by the first
  // kernel (which also zeroes the H histograms in use), `keys` and the histogram counts by the second; what an earlier call left
  // behind in the array is never looked at.
  token_qsum_kernel<<<dim3(n_chunks, g.H), 256, 0, st>>>((const __nv_bfloat16 *)q, part, hist1, g);
  token_probe_kernel<<<dim3((unsigned)((g.N + kTokTile - 1) / kTokTile), g.H), 256, 0, st>>>((const __nv_bfloat16 *)k, part, keys, hist1,
                                                                                           g, n_chunks);
  token_topk_kernel<<<g.H, 1024, 0, st>>>(keys, hist1, idx, g.N, K);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return noalloc_fail(err_buf, err_len, SAF3R_ERR_CUDA, std::string("token probe launch: ") + cudaGetErrorString(e));
  return SAF3R_OK;
}

saf3r_status saf3r_token_set_attn(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape,
                                  const int32_t *idx, int32_t K, void *ws, size_t ws_bytes, void *out, int out_is_fp32, float *lse,
                                  void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  const SelGeom g = make_geom(shape);
  if (K < 1 || K > g.N) return fail(ctx, SAF3R_ERR_INVALID_ARG, "token set: need 1 <= K <= N");
  if (!q || !k || !v || !ws || !idx || !out) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)k | (uintptr_t)v | (uintptr_t)ws) & 15) return fail(ctx, SAF3R_ERR_INVALID_ARG, "k/v/workspace must be 16-byte aligned");
  const TokWs w = tok_ws(g, K);
  if (ws_bytes < w.attn_total) return fail(ctx, SAF3R_ERR_CAPACITY, "workspace too small (saf3r_token_query_sizes)");
  cudaStream_t st = (cudaStream_t)stream_;
  __nv_bfloat16 *kc = (__nv_bfloat16 *)((uint8_t *)ws + w.kc), *vc = (__nv_bfloat16 *)((uint8_t *)ws + w.vc);
  token_gather_kernel<<<dim3((K + 31) / 32, g.H, 2), 256, 0, st>>>((const __nv_bfloat16 *)k, (const __nv_bfloat16 *)v, idx, kc, vc, g, K);
  ctx->launches += 1;
  CU_CHECK(cudaGetLastError());
  const KvGeom kv{K, (int64_t)K * 64, 64};
  return attn_common(ctx, q, kc, vc, shape, nullptr, out, out_is_fp32, lse, stream_, &kv);
}

saf3r_status saf3r_nmse_accumulate(saf3r_ctx *ctx, const void *o_full, const void *o_sparse, const saf3r_shape *shape, int is_fp32,
                                   double *num_den, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!o_full || !o_sparse || !num_den) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)o_full | (uintptr_t)o_sparse) & 15) return fail(ctx, SAF3R_ERR_INVALID_ARG, "outputs must be 16-byte aligned");
  const SelGeom g = make_geom(shape);
  nmse_kernel<<<dim3(4 * ctx->sm_count / (g.H < 4 ? g.H : 4) + 1, g.H), 256, 0, (cudaStream_t)stream_>>>(
      (const uint8_t *)o_full, (const uint8_t *)o_sparse, g.N, g.stride_head, g.stride_token, is_fp32 ? 1 : 0, num_den, num_den + g.H);
  ctx->launches += 1;
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

// ------------------------------------------------------------------------------------------------ token-wise per-frame Top-K (NEXT-2 iii)
struct TokTopkWs { size_t rn, keys, total; int64_t ld; int strips; };
static TokTopkWs toktopk_ws(int64_t N) {
  TokTopkWs w;
  const int64_t nb = (N + 127) / 128;
  w.ld = nb * 128;
  const int64_t strip_bytes = 128 * w.ld * 4;
  int64_t strips = (48ll << 20) / strip_bytes;  // q-tiles per launch pair: keep the key strip L2-sized
  if (strips < 1) strips = 1;
  if (strips > 8) strips = 8;
  if (strips > nb) strips = nb;
  w.strips = (int)strips;
  size_t off = 0;
  w.rn = off; off = align256(off + (size_t)N * sizeof(float));
  w.keys = off; off = align256(off + (size_t)strips * strip_bytes);
  w.total = off;
  return w;
}
static int64_t toktopk_max_tiles(const SelGeom &g, int K) {
  const int64_t per_frame = i64min(g.T, (int64_t)g.B * K);  // distinct keys a q-tile of B queries can pick in one frame
  return (int64_t)g.NB * (((int64_t)g.S * per_frame + g.B - 1) / g.B);
}
static const char *validate_toktopk(const saf3r_shape *shape, int K) {
  if (const char *m = validate_shape(shape, false)) return m;
  if (K < 1 || K > shape->tokens_per_frame) return "token-wise Top-K: need 1 <= K <= tokens_per_frame";
  return nullptr;
}

saf3r_status saf3r_token_topk_query_sizes(const saf3r_shape *shape, int32_t K, size_t *select_ws, int64_t *idx_entries, int64_t *max_tiles) {
  if (validate_toktopk(shape, K)) return SAF3R_ERR_INVALID_ARG;
  if (unsupported_shape(shape)) return SAF3R_ERR_UNSUPPORTED;
  const SelGeom g = make_geom(shape);
  if (select_ws) *select_ws = toktopk_ws(g.N).total;
  if (idx_entries) *idx_entries = g.N * g.S * K;
  if (max_tiles) *max_tiles = toktopk_max_tiles(g, K);
  return SAF3R_OK;
}

saf3r_status saf3r_token_topk_select(saf3r_ctx *ctx, const void *feat, const saf3r_shape *shape, int32_t K, void *ws, size_t ws_bytes,
                                     int32_t *idx, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_toktopk(shape, K)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!feat || !ws || !idx) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (shape->stride_token < 64 || shape->stride_token % 8 || ((uintptr_t)feat & 15))
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "features: 16-byte aligned, stride_token a multiple of 8 elements and >= head_dim");
  SelGeom g = make_geom(shape);
  g.H = 1; g.B = 128; g.NB = (int32_t)((g.N + 127) / 128);
  g.stride_head = g.N * g.stride_token;
  const TokTopkWs w = toktopk_ws(g.N);
  if (ws_bytes < w.total) return fail(ctx, SAF3R_ERR_CAPACITY, "workspace too small (saf3r_token_topk_query_sizes)");
  CUtensorMap mf;
  saf3r_status s;
  if ((s = get_map(ctx, feat, g, &mf)) != SAF3R_OK) return s;
  cudaStream_t st = (cudaStream_t)stream_;
  float *rn = (float *)((uint8_t *)ws + w.rn);
  uint32_t *keys = (uint32_t *)((uint8_t *)ws + w.keys);
  feat_rnorm_kernel<<<(unsigned)((g.N + 31) / 32), 256, 0, st>>>((const __nv_bfloat16 *)feat, g.N, g.stride_token, rn);
  ctx->launches += 1;
  for (int q0 = 0; q0 < g.NB; q0 += w.strips) {
    const int nq = g.NB - q0 < w.strips ? g.NB - q0 : w.strips;
    token_sim_kernel<<<dim3(g.NB, nq), 128, kSimSmem, st>>>(mf, rn, keys, g.N, w.ld, q0);
    const int64_t warps = (int64_t)nq * 128 * g.S;
    token_frame_topk_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(keys, w.ld, (int64_t)q0 * 128, nq * 128, g.N, g.S, g.T, K, idx);
    ctx->launches += 2;
  }
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

static saf3r_status toklists_common(saf3r_ctx *ctx, const saf3r_shape *shape, int K, const int32_t *idx, int64_t *tile_ptr,
                                    const saf3r_token_lists *lists, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_toktopk(shape, K)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!idx || !tile_ptr || (lists && (!lists->key_idx || !lists->mask))) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  const SelGeom g = make_geom(shape);
  const size_t sm = 2 * (size_t)((g.T + 31) / 32) * sizeof(uint32_t);
  if (sm > 48 * 1024) return fail(ctx, SAF3R_ERR_UNSUPPORTED, "tokens_per_frame too large for the union kernel");
  cudaStream_t st = (cudaStream_t)stream_;
  if (!lists) {
    token_union_kernel<false><<<g.NB, 256, sm, st>>>(idx, g.N, g.S, g.T, K, g.B, tile_ptr, nullptr, nullptr, 0);
    scan_row_ptr_kernel<<<1, 1024, 0, st>>>(tile_ptr, g.NB);
    ctx->launches += 2;
  } else {
    CU_CHECK(cudaMemsetAsync(lists->mask, 0, (size_t)lists->capacity_tiles * g.B * (g.B / 32) * sizeof(uint32_t), st));
    token_union_kernel<true><<<g.NB, 256, sm, st>>>(idx, g.N, g.S, g.T, K, g.B, tile_ptr, lists->key_idx, lists->mask, lists->capacity_tiles);
    ctx->launches += 1;
  }
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

saf3r_status saf3r_token_lists_count(saf3r_ctx *ctx, const saf3r_shape *shape, int32_t K, const int32_t *idx, int64_t *tile_ptr, void *stream) {
  return toklists_common(ctx, shape, K, idx, tile_ptr, nullptr, stream);
}

saf3r_status saf3r_token_lists_fill(saf3r_ctx *ctx, const saf3r_shape *shape, int32_t K, const int32_t *idx, const saf3r_token_lists *lists,
                                    void *stream) {
  if (!lists) return fail(ctx, SAF3R_ERR_INVALID_ARG, "lists is null");
  return toklists_common(ctx, shape, K, idx, lists->tile_ptr, lists, stream);
}

saf3r_status saf3r_token_lists_attn(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape,
                                    const saf3r_token_lists *lists, void *out, int out_is_fp32, float *lse, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!q || !k || !v || !out || !lists || !lists->tile_ptr || !lists->key_idx || !lists->mask)
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (lists->capacity_tiles < 0) return fail(ctx, SAF3R_ERR_INVALID_ARG, "token lists: capacity_tiles must be >= 0");
  if (((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out) & 15) return fail(ctx, SAF3R_ERR_INVALID_ARG, "q/k/v/out must be 16-byte aligned");
  const SelGeom g = make_geom(shape);
  CUtensorMap mq;
  saf3r_status s;
  if ((s = get_map(ctx, q, g, &mq)) != SAF3R_OK) return s;
  AttnParams p;
  memset(&p, 0, sizeof p);
  p.out = out; p.lse = lse;
  p.out_stride_head = shape->stride_head; p.out_stride_token = shape->stride_token;
  p.N = (int32_t)g.N; p.NB = g.NB; p.H = g.H; p.N_kv = (int32_t)g.N; p.NB_kv = g.NB;
  p.out_fp32 = out_is_fp32 ? 1 : 0;
  p.scale_log2 = (float)(1.4426950408889634 / sqrt((double)shape->head_dim));
  p.head_order = nullptr;
  p.tile_ptr = lists->tile_ptr; p.key_idx = lists->key_idx; p.mask = lists->mask; p.capacity_tiles = lists->capacity_tiles;
  p.k_base = (const __nv_bfloat16 *)k; p.v_base = (const __nv_bfloat16 *)v;
  p.kv_stride_head = g.stride_head; p.kv_stride_token = g.stride_token;
  cudaStream_t st = (cudaStream_t)stream_;
  float *slot = ctx->kmax_ring + (size_t)(ctx->kmax_next++ % kKmaxSlots) * kKmaxSlotFloats;
  CU_CHECK(cudaMemsetAsync(slot, 0, sizeof(float) * g.H, st));
  knorm_kernel<<<dim3((unsigned)((g.N + kKnormRows - 1) / kKnormRows), g.H), 256, 0, st>>>((const __nv_bfloat16 *)k, g.N, g.stride_head, g.stride_token, slot,
                                                                                          nullptr, g.NB, reinterpret_cast<uint8_t *>(slot + SAF3R_MAX_HEADS));
  p.kmax = slot;
  dim3 grid(g.NB, g.H);
  if (g.B == 128)
    saf3r_attn_kernel<128, true><<<grid, kAttnThreads, AttnSmem<128>::kTotal, st>>>(mq, mq, mq, p);
  else
    saf3r_attn_kernel<64, true><<<grid, kAttnThreads, AttnSmem<64>::kTotal, st>>>(mq, mq, mq, p);
  ctx->launches += 2;
  CU_CHECK(cudaGetLastError());
  return SAF3R_OK;
}

// ------------------------------------------------------------------------------------------------ static broadcast (NEXT-4)
struct BcastWs { size_t kc, vc, lse0, total; };
static BcastWs bcast_ws(const SelGeom &g) {
  BcastWs w;
  size_t off = 0;
  w.kc = off; off = align256(off + (size_t)g.H * g.T * 64 * 2);
  w.vc = off; off = align256(off + (size_t)g.H * g.T * 64 * 2);
  w.lse0 = off; off = align256(off + (size_t)g.H * g.T * sizeof(float));
  w.total = off;
  return w;
}

saf3r_status saf3r_static_broadcast_workspace_bytes(const saf3r_shape *shape, size_t *bytes) {
  if (validate_shape(shape, false) || !bytes) return SAF3R_ERR_INVALID_ARG;
  if (unsupported_shape(shape)) return SAF3R_ERR_UNSUPPORTED;
  *bytes = bcast_ws(make_geom(shape)).total;
  return SAF3R_OK;
}

saf3r_status saf3r_static_broadcast_attn(saf3r_ctx *ctx, const void *q, const void *k, const void *v, const saf3r_shape *shape, void *ws,
                                         size_t ws_bytes, void *out, int out_is_fp32, float *lse, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape, true)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  if (!q || !k || !v || !ws || !out) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  if (((uintptr_t)q | (uintptr_t)k | (uintptr_t)v | (uintptr_t)out | (uintptr_t)ws) & 15)
    return fail(ctx, SAF3R_ERR_INVALID_ARG, "q/k/v/out/workspace must be 16-byte aligned");
  const SelGeom g = make_geom(shape);
  const BcastWs w = bcast_ws(g);
  if (ws_bytes < w.total) return fail(ctx, SAF3R_ERR_CAPACITY, "workspace too small (saf3r_static_broadcast_workspace_bytes)");
  cudaStream_t st = (cudaStream_t)stream_;
  __nv_bfloat16 *kc = (__nv_bfloat16 *)((uint8_t *)ws + w.kc), *vc = (__nv_bfloat16 *)((uint8_t *)ws + w.vc);
  float *lse0 = (float *)((uint8_t *)ws + w.lse0);
  frame_mean_kernel<<<dim3((g.T + 31) / 32, g.H, 2), 256, 0, st>>>((const __nv_bfloat16 *)k, (const __nv_bfloat16 *)v, kc, vc, g);
  ctx->launches += 1;
  CU_CHECK(cudaGetLastError());
  // frame 0's rows of `out` = dense attention of (Q0, K0, vbar); the query geometry is the caller's with a single frame
  saf3r_shape one = *shape;
  one.num_frames = 1;
  const KvGeom kv{g.T, (int64_t)g.T * 64, 64};
  saf3r_status s = attn_common(ctx, q, kc, vc, &one, nullptr, out, out_is_fp32, lse ? lse0 : nullptr, stream_, &kv);
  if (s != SAF3R_OK) return s;
  if (g.S > 1 || lse) {
    const int elem = out_is_fp32 ? 4 : 2, rows = 256 / (4 * elem);
    frame_broadcast_kernel<<<dim3((g.T + rows - 1) / rows, g.S, g.H), 256, 0, st>>>((uint8_t *)out, lse, lse0, g, shape->stride_head,
                                                                                   shape->stride_token, elem);
    ctx->launches += 1;
    CU_CHECK(cudaGetLastError());
  }
  return SAF3R_OK;
}

// saf3r_layer_host pipelines the layer over groups of heads (heads are independent): the host->device copy of
// group g+1 runs under the select + attention of group g, and the device->host copy of group g under the compute of group
// g+1 (separate copy engines), on ctx-owned side streams forked from / joined to the caller's stream with events.
constexpr int kHostGroups = 9, kHostStreams = 3;
struct HostGroup { int h0, hn; size_t ws, row_ptr, col_idx; int64_t entries; };
struct HostLayout {
  size_t q, k, v, out, total;
  int n_groups;
  HostGroup grp[kHostGroups];
};
static SelGeom sub_geom(const SelGeom &g, int hn) {
  SelGeom s = g;
  s.H = hn;
  return s;
}
static HostLayout host_layout(const SelGeom &g, const saf3r_head_cfg *cfg) {
  HostLayout l;
  const size_t t = align256((size_t)g.H * g.N * 64 * 2);
  size_t off = 0;
  l.q = off; off += t;
  l.k = off; off += t;
  l.v = off; off += t;
  l.out = off; off += t;
  l.n_groups = g.H < kHostGroups ? g.H : kHostGroups;
  int h0 = 0;
  for (int i = 0; i < l.n_groups; ++i) {
    HostGroup &gr = l.grp[i];
    gr.h0 = h0;
    // when there are more heads than groups the LAST group is a single head: what follows the last host->device copy (that
    // group's select + attention + device->host copy) is exposed, so it is kept as short as the split allows
    const int tail = g.H > l.n_groups ? 1 : 0;
    gr.hn = (tail && i == l.n_groups - 1) ? g.H - h0 : (g.H - tail - h0 + (l.n_groups - tail - i) - 1) / (l.n_groups - tail - i);
    h0 += gr.hn;
    const SelGeom sg = sub_geom(g, gr.hn);
    gr.ws = off; off += ws_layout(sg).total;
    gr.row_ptr = off; off = align256(off + ((size_t)gr.hn * g.NB + 1) * 8);
    gr.entries = total_entries(sg, cfg + gr.h0);
    gr.col_idx = off; off = align256(off + (size_t)(gr.entries > 0 ? gr.entries : 1) * 4);
  }
  l.total = off;
  return l;
}

saf3r_status saf3r_layer_host_scratch_bytes(const saf3r_shape *shape, const saf3r_head_cfg *cfg, size_t *bytes) {
  if (validate_shape(shape, false) || !cfg || !bytes) return SAF3R_ERR_INVALID_ARG;
  if (unsupported_shape(shape)) return SAF3R_ERR_UNSUPPORTED;
  const SelGeom g = make_geom(shape);
  if (validate_cfg(g, cfg)) return SAF3R_ERR_INVALID_ARG;
  *bytes = host_layout(g, cfg).total;
  return SAF3R_OK;
}

saf3r_status saf3r_layer_host(saf3r_ctx *ctx, const void *qh, const void *kh, const void *vh, const saf3r_shape *shape_in,
                              const saf3r_head_cfg *cfg, void *scratch, size_t scratch_bytes, void *out_host, void *stream_) {
  if (!ctx) return SAF3R_ERR_INVALID_ARG;
  if (ctx->sticky_cuda) return SAF3R_ERR_CUDA;
  if (const char *m = validate_shape(shape_in, false)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (const char *m = unsupported_shape(shape_in)) return fail(ctx, SAF3R_ERR_UNSUPPORTED, m);
  saf3r_shape shape = *shape_in;
  shape.stride_token = 64;
  shape.stride_head = (int64_t)shape.num_frames * shape.tokens_per_frame * 64;
  const SelGeom g = make_geom(&shape);
  if (const char *m = validate_cfg(g, cfg)) return fail(ctx, SAF3R_ERR_INVALID_ARG, m);
  if (!qh || !kh || !vh || !scratch || !out_host) return fail(ctx, SAF3R_ERR_INVALID_ARG, "null pointer argument");
  const HostLayout l = host_layout(g, cfg);
  if (scratch_bytes < l.total) return fail(ctx, SAF3R_ERR_CAPACITY, "scratch too small (see saf3r_layer_host_scratch_bytes)");
  if (!ctx->side[0]) {
    for (auto &sd : ctx->side) CU_CHECK(cudaStreamCreateWithFlags(&sd, cudaStreamNonBlocking));
    CU_CHECK(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
    for (auto &e : ctx->ev_join) CU_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  cudaStream_t st = (cudaStream_t)stream_;
  uint8_t *sb = (uint8_t *)scratch;
  const size_t head_bytes = (size_t)g.N * 64 * 2;
  CU_CHECK(cudaEventRecord(ctx->ev_fork, st));
  const int n_streams = l.n_groups < kHostStreams ? l.n_groups : kHostStreams;
  for (int i = 0; i < n_streams; ++i) CU_CHECK(cudaStreamWaitEvent(ctx->side[i], ctx->ev_fork, 0));
  for (int i = 0; i < l.n_groups; ++i) {
    const HostGroup &gr = l.grp[i];
    cudaStream_t ss = ctx->side[i % kHostStreams];
    const size_t o = (size_t)gr.h0 * head_bytes, nb = (size_t)gr.hn * head_bytes;
    CU_CHECK(cudaMemcpyAsync(sb + l.q + o, (const uint8_t *)qh + o, nb, cudaMemcpyHostToDevice, ss));
    CU_CHECK(cudaMemcpyAsync(sb + l.k + o, (const uint8_t *)kh + o, nb, cudaMemcpyHostToDevice, ss));
    CU_CHECK(cudaMemcpyAsync(sb + l.v + o, (const uint8_t *)vh + o, nb, cudaMemcpyHostToDevice, ss));
    saf3r_shape sub = shape;
    sub.num_heads = gr.hn;
    saf3r_lists lists{(int64_t *)(sb + gr.row_ptr), (int32_t *)(sb + gr.col_idx), gr.entries > 0 ? gr.entries : 1};
    saf3r_status s = saf3r_select(ctx, sb + l.q + o, sb + l.k + o, &sub, cfg + gr.h0, sb + gr.ws, ws_layout(sub_geom(g, gr.hn)).total,
                                  &lists, ss);
    if (s != SAF3R_OK) return s;
    s = saf3r_sparse_attn(ctx, sb + l.q + o, sb + l.k + o, sb + l.v + o, &sub, &lists, sb + l.out + o, 0, nullptr, ss);
    if (s != SAF3R_OK) return s;
    CU_CHECK(cudaMemcpyAsync((uint8_t *)out_host + o, sb + l.out + o, nb, cudaMemcpyDeviceToHost, ss));
  }
  for (int i = 0; i < n_streams; ++i) {
    CU_CHECK(cudaEventRecord(ctx->ev_join[i], ctx->side[i]));
    CU_CHECK(cudaStreamWaitEvent(st, ctx->ev_join[i], 0));
  }
  return SAF3R_OK;
}

}  // extern "C"
