// Online pattern adaptation at block granularity (steps a-1..a-3 of DESIGN.md):
//   pool_kernel      Q,K bf16 -> Qtilde,Ktilde fp32 block means (HBM-bound stream)
//   qbar_kernel      qbar = (1/N) sum_t q_t from the pooled block means
//   rowlen_kernel    closed-form list length of every (head, q-block) row;  scan_kernel -> row_ptr
//   probe_kernel     p[J] = qbar . Ktilde_J / sqrt(D), top-n -> one shared list per QUERY_PROBE head
//   select_kernel    per (head, q-block): closed-form emit, probe-list copy, or score row + top-n / per-frame top-k
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "saf3r.h"

namespace saf3r {

struct SelGeom {
  int32_t S, T, H, B, NB;
  int64_t N;
  int64_t stride_head, stride_token;
};

struct HeadCfgArray {
  saf3r_head_cfg c[SAF3R_MAX_HEADS];
};

__host__ __device__ inline int64_t i64min(int64_t a, int64_t b) { return a < b ? a : b; }
__host__ __device__ inline int64_t i64max(int64_t a, int64_t b) { return a > b ? a : b; }

// Number of candidate k-blocks of frame g for PER_FRAME scope: C_g = {J : floor(J*B/T) = g} = [ceil(gT/B), ceil((g+1)T/B) - 1].
__host__ __device__ inline void frame_candidates(const SelGeom &g, int64_t f, int64_t &lo, int64_t &hi) {
  lo = (f * g.T + g.B - 1) / g.B;
  hi = i64min(((f + 1) * g.T + g.B - 1) / g.B - 1, (int64_t)g.NB - 1);
}

// Closed-form rows (DENSE, UNIFORM_STRIDE, STATIC): visit the kept k-blocks of q-block I in ascending order.
// F is called as f(J).  Returns the count.  Shared by the host sizing code and the device emitters.
template <class F>
__host__ __device__ inline int64_t closed_form_row(const SelGeom &g, const saf3r_head_cfg &c, int64_t I, F &&f) {
  const int64_t NB = g.NB, T = g.T, B = g.B, N = g.N;
  int64_t cnt = 0;
  if (c.type == SAF3R_HEAD_DENSE) {
    for (int64_t J = 0; J < NB; ++J) { f(J); ++cnt; }
  } else if (c.type == SAF3R_HEAD_UNIFORM_STRIDE) {
    if (c.stride >= 1) {
      for (int64_t J = c.offset; J < NB; J += c.stride) { f(J); ++cnt; }
    } else {
      int64_t prev = -1;
      for (int64_t i = 0; i < c.keep_blocks; ++i) {
        int64_t J = (i * NB) / c.keep_blocks;
        if (J != prev) { f(J); ++cnt; prev = J; }
      }
    }
  } else if (c.type == SAF3R_HEAD_STATIC) {
    const int64_t t0 = I * B, t1 = i64min(t0 + B, N);
    const int64_t f0 = t0 / T, f1 = (t1 - 1) / T;
    if (c.static_mode == SAF3R_STATIC_ANCHOR) {
      const int64_t a = c.anchor_frame;
      for (int64_t J = (a * T) / B; J <= ((a + 1) * T - 1) / B; ++J) { f(J); ++cnt; }
    } else if (c.static_mode == SAF3R_STATIC_FRAME_LOCAL) {
      for (int64_t J = (f0 * T) / B; J <= ((f1 + 1) * T - 1) / B; ++J) { f(J); ++cnt; }
    } else {
      // POSITION_BAND: in-frame position intervals (at most two disjoint ones), replicated in every frame
      const int64_t r = c.band_radius;
      int64_t lo[2], hi[2];
      int ni;
      if (f1 == f0) {
        lo[0] = i64max(0, t0 - f0 * T - r); hi[0] = i64min(T - 1, (t1 - 1) - f0 * T + r); ni = 1;
      } else if (f1 - f0 >= 2) {
        lo[0] = 0; hi[0] = T - 1; ni = 1;                     // a whole frame lies inside the q-block
      } else {
        const int64_t loA = i64max(0, t0 - f0 * T - r);      // tail of frame f0: positions [loA, T-1]
        const int64_t hiB = i64min(T - 1, (t1 - 1) - f1 * T + r);  // head of frame f1: positions [0, hiB]
        if (hiB + 1 >= loA) { lo[0] = 0; hi[0] = T - 1; ni = 1; }
        else { lo[0] = 0; hi[0] = hiB; lo[1] = loA; hi[1] = T - 1; ni = 2; }
      }
      int64_t last = -1;
      for (int64_t fr = 0; fr < g.S; ++fr)
        for (int q = 0; q < ni; ++q) {
          int64_t a = i64max((fr * T + lo[q]) / B, last + 1), b = (fr * T + hi[q]) / B;
          for (int64_t J = a; J <= b; ++J) { f(J); ++cnt; }
          if (b > last) last = b;
        }
    }
  }
  return cnt;
}

// List length of a row (any head type); a closed form of (shape, cfg).
__host__ __device__ inline int64_t row_length(const SelGeom &g, const saf3r_head_cfg &c, int64_t I) {
  if (c.type == SAF3R_HEAD_QUERY_PROBE_TOPK || (c.type == SAF3R_HEAD_BLOCK_TOPK && c.topk_scope == SAF3R_SCOPE_GLOBAL))
    return i64min(c.keep_blocks, g.NB);
  if (c.type == SAF3R_HEAD_BLOCK_TOPK) {
    int64_t cnt = 0;
    for (int64_t f = 0; f < g.S; ++f) {
      int64_t lo, hi;
      frame_candidates(g, f, lo, hi);
      cnt += i64min(c.topk_per_frame, i64max(0, hi - lo + 1));
    }
    return cnt;
  }
  if (c.type == SAF3R_HEAD_DENSE) return g.NB;
  if (c.type == SAF3R_HEAD_UNIFORM_STRIDE && c.stride >= 1) return (g.NB - c.offset + c.stride - 1) / c.stride;
  return closed_form_row(g, c, I, [](int64_t) {});
}

// ------------------------------------------------------------------------------------------------ pool
// grid (NB, H, 2): z = 0 pools Q, z = 1 pools K.  256 threads: 8 threads per token row (16 B each), 32 rows per pass.
// flags[h] bit0: pool Q, bit1: pool K, bit2: cosine (L2-normalise each token first).
struct PoolFlags { uint8_t f[SAF3R_MAX_HEADS]; };

__global__ void __launch_bounds__(256) pool_kernel(const __nv_bfloat16 *__restrict__ q, const __nv_bfloat16 *__restrict__ k,
                                                   float *__restrict__ qt, float *__restrict__ kt, SelGeom g, PoolFlags flags) {
  const int J = blockIdx.x, h = blockIdx.y, which = blockIdx.z;
  const uint8_t fl = flags.f[h];
  if (!((fl >> which) & 1)) return;
  const bool cosine = (fl >> 2) & 1;
  const __nv_bfloat16 *src = (which ? k : q) + (int64_t)h * g.stride_head;
  float *dst = (which ? kt : qt) + ((int64_t)h * g.NB + J) * 64;
  const int64_t t0 = (int64_t)J * g.B;
  const int cnt = (int)i64min(g.B, g.N - t0);
  const int sub = threadIdx.x & 7, rg = threadIdx.x >> 3;  // 16-byte chunk within the row, row group
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  constexpr int kMaxPass = 4;  // B <= 128
  uint4 raw[kMaxPass];
#pragma unroll
  for (int ps = 0; ps < kMaxPass; ++ps) {
    const int r = ps * 32 + rg;
    raw[ps] = make_uint4(0, 0, 0, 0);
    if (r < cnt) raw[ps] = __ldg(reinterpret_cast<const uint4 *>(src + (t0 + r) * g.stride_token) + sub);
  }
#pragma unroll
  for (int ps = 0; ps < kMaxPass; ++ps) {
    const uint32_t w[4] = {raw[ps].x, raw[ps].y, raw[ps].z, raw[ps].w};
    float v[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      v[2 * i] = __uint_as_float(w[i] << 16);
      v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
    float inv = 1.f;
    if (cosine) {
      float ss = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) ss = fmaf(v[i], v[i], ss);
      ss += __shfl_xor_sync(0xffffffffu, ss, 1);
      ss += __shfl_xor_sync(0xffffffffu, ss, 2);
      ss += __shfl_xor_sync(0xffffffffu, ss, 4);
      const float nrm = sqrtf(ss);
      inv = nrm < 1e-20f ? 0.f : 1.f / nrm;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = fmaf(v[i], inv, acc[i]);
  }
  __shared__ float part[32][65];
#pragma unroll
  for (int i = 0; i < 8; ++i) part[rg][sub * 8 + i] = acc[i];
  __syncthreads();
  if (threadIdx.x < 64) {
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < 32; ++r) s += part[r][threadIdx.x];
    dst[threadIdx.x] = s / (float)cnt;
  }
}

// ------------------------------------------------------------------------------------------------ qbar
// grid (H); 256 threads = 4 groups x 64 dims.  qbar[d] = (1/N) sum_J c_J * Qtilde[J][d].
__global__ void __launch_bounds__(256) qbar_kernel(const float *__restrict__ qt, float *__restrict__ qbar, SelGeom g,
                                                   HeadCfgArray cfg) {
  const int h = blockIdx.x;
  if (cfg.c[h].type != SAF3R_HEAD_QUERY_PROBE_TOPK) return;
  const int d = threadIdx.x & 63, grp = threadIdx.x >> 6;
  float s = 0.f;
  for (int J = grp; J < g.NB; J += 4) {
    const float cnt = (float)i64min(g.B, g.N - (int64_t)J * g.B);
    s = fmaf(qt[((int64_t)h * g.NB + J) * 64 + d], cnt, s);
  }
  __shared__ float part[4][64];
  part[grp][d] = s;
  __syncthreads();
  if (grp == 0) qbar[h * 64 + d] = (part[0][d] + part[1][d] + part[2][d] + part[3][d]) / (float)g.N;
}

// ------------------------------------------------------------------------------------------------ row lengths + scan
__global__ void rowlen_kernel(int32_t *__restrict__ rowlen, SelGeom g, HeadCfgArray cfg) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= (int64_t)g.H * g.NB) return;
  const int h = (int)(r / g.NB);
  rowlen[r] = (int32_t)row_length(g, cfg.c[h], r % g.NB);
}

// single CTA, 1024 threads: exclusive scan of rowlen[n] into row_ptr[n+1] (int64)
__global__ void __launch_bounds__(1024) scan_kernel(const int32_t *__restrict__ rowlen, int64_t *__restrict__ row_ptr, int64_t n) {
  __shared__ int64_t sums[1024];
  const int64_t per = (n + 1023) / 1024;
  const int64_t a = i64min(n, threadIdx.x * per), b = i64min(n, a + per);
  int64_t s = 0;
  for (int64_t i = a; i < b; ++i) s += rowlen[i];
  sums[threadIdx.x] = s;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {  // Hillis-Steele inclusive scan
    int64_t v = threadIdx.x >= off ? sums[threadIdx.x - off] : 0;
    __syncthreads();
    sums[threadIdx.x] += v;
    __syncthreads();
  }
  int64_t run = threadIdx.x ? sums[threadIdx.x - 1] : 0;
  for (int64_t i = a; i < b; ++i) {
    row_ptr[i] = run;
    run += rowlen[i];
  }
  if (threadIdx.x == 1023) row_ptr[n] = sums[1023];
}

// ------------------------------------------------------------------------------------------------ warp-level top-n
// Order-preserving key: larger float <-> larger key; -0 is folded onto +0 so that ties follow the float comparison.
__device__ __forceinline__ uint32_t score_key(float s) {
  uint32_t u = __float_as_uint(s);
  if (u == 0x80000000u) u = 0u;
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// One warp: keep the n largest of s[0..NB) under (score desc, index asc); write their indices ascending to out.
// hist: 256 uint32 of shared memory private to the warp.  Radix-select the n-th largest key (4 passes of 8 bits),
// then an ordered compaction: {key > tau} plus the first `need` (by index) of {key == tau}.
__device__ inline void warp_topn_emit(const float *s, int NB, int n, int32_t *out, uint32_t *hist) {
  const int lane = threadIdx.x & 31;
  uint32_t prefix = 0, mask = 0;
  int need = n;
  for (int shift = 24; shift >= 0; shift -= 8) {
    for (int i = lane; i < 256; i += 32) hist[i] = 0;
    __syncwarp();
    for (int j = lane; j < NB; j += 32) {
      const uint32_t key = score_key(s[j]);
      if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
    }
    __syncwarp();
    // lane L owns buckets 255-8L .. 248-8L (descending); find the bucket where the running count reaches `need`
    uint32_t loc[8], tot = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { loc[i] = hist[255 - 8 * lane - i]; tot += loc[i]; }
    uint32_t inc = tot;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      uint32_t v = __shfl_up_sync(0xffffffffu, inc, off);
      if (lane >= off) inc += v;
    }
    const uint32_t exc = inc - tot;
    const uint32_t hit = __ballot_sync(0xffffffffu, inc >= (uint32_t)need);
    const int src = __ffs(hit) - 1;
    int bucket = 0, above = 0;
    if (lane == src) {
      uint32_t run = exc;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (run + loc[i] >= (uint32_t)need) { bucket = 255 - 8 * lane - i; above = (int)run; break; }
        run += loc[i];
      }
    }
    bucket = __shfl_sync(0xffffffffu, bucket, src);
    above = __shfl_sync(0xffffffffu, above, src);
    need -= above;
    prefix |= (uint32_t)bucket << shift;
    mask |= 255u << shift;
    __syncwarp();
  }
  const uint32_t tau = prefix;  // key of the n-th largest score; take `need` of the elements equal to it, lowest index first
  int written = 0, eq_seen = 0;
  const uint32_t lt = (1u << lane) - 1u;
  for (int j0 = 0; j0 < NB; j0 += 32) {
    const int j = j0 + lane;
    const uint32_t key = j < NB ? score_key(s[j]) : 0u;
    const bool gt = j < NB && key > tau, eq = j < NB && key == tau;
    const uint32_t eqb = __ballot_sync(0xffffffffu, eq);
    const bool take = gt || (eq && eq_seen + __popc(eqb & lt) < need);
    const uint32_t tb = __ballot_sync(0xffffffffu, take);
    if (take) out[written + __popc(tb & lt)] = j;
    written += __popc(tb);
    eq_seen += __popc(eqb);
  }
}

// One warp: per-frame top-k (PER_FRAME scope): in every frame's candidate range keep the kf best; ascending output.
__device__ inline void warp_per_frame_emit(const float *s, const SelGeom &g, int kf, int32_t *out) {
  const int lane = threadIdx.x & 31;
  int base = 0;
  for (int f0 = 0; f0 < g.S; f0 += 32) {
    const int f = f0 + lane;
    int64_t lo = 0, hi = -1;
    if (f < g.S) frame_candidates(g, f, lo, hi);
    const int m = (int)i64max(0, hi - lo + 1);
    const int keep = m < kf ? m : kf;
    int inc = keep;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      int v = __shfl_up_sync(0xffffffffu, inc, off);
      if (lane >= off) inc += v;
    }
    int pos = base + inc - keep;
    for (int a = 0; a < m; ++a) {
      const float sa = s[lo + a];
      int rank = 0;
      for (int b = 0; b < m; ++b) {
        const float sb = s[lo + b];
        rank += (sb > sa) || (sb == sa && b < a);
      }
      if (rank < kf) out[pos++] = (int32_t)(lo + a);
    }
    base += __shfl_sync(0xffffffffu, inc, 31);
  }
}

// ------------------------------------------------------------------------------------------------ probe
// grid (H), 256 threads, dynamic smem: NB floats + 256 uint32.  Writes the shared list of a QUERY_PROBE head to
// probe_list[h][0..n).
__global__ void __launch_bounds__(256) probe_kernel(const float *__restrict__ kt, const float *__restrict__ qbar,
                                                    int32_t *__restrict__ probe_list, SelGeom g, HeadCfgArray cfg) {
  const int h = blockIdx.x;
  if (cfg.c[h].type != SAF3R_HEAD_QUERY_PROBE_TOPK) return;
  extern __shared__ float sm[];
  float *s = sm;
  uint32_t *hist = reinterpret_cast<uint32_t *>(sm + g.NB);
  __shared__ float qb[64];
  if (threadIdx.x < 64) qb[threadIdx.x] = qbar[h * 64 + threadIdx.x];
  __syncthreads();
  for (int J = threadIdx.x; J < g.NB; J += blockDim.x) {
    const float4 *kr = reinterpret_cast<const float4 *>(kt + ((int64_t)h * g.NB + J) * 64);
    float acc = 0.f;
#pragma unroll
    for (int d4 = 0; d4 < 16; ++d4) {
      const float4 kv = __ldg(kr + d4);
      acc = fmaf(qb[4 * d4], kv.x, acc);
      acc = fmaf(qb[4 * d4 + 1], kv.y, acc);
      acc = fmaf(qb[4 * d4 + 2], kv.z, acc);
      acc = fmaf(qb[4 * d4 + 3], kv.w, acc);
    }
    s[J] = acc * 0.125f;
  }
  __syncthreads();
  if (threadIdx.x < 32) warp_topn_emit(s, g.NB, (int)i64min(cfg.c[h].keep_blocks, g.NB), probe_list + (int64_t)h * g.NB, hist);
}

// ------------------------------------------------------------------------------------------------ select
// grid (ceil(NB/R), H), 256 threads (8 warps), R <= 8 rows per CTA.  dynamic smem: R*NB floats (scores) + R*64 floats
// (Qtilde rows) + 8*256 uint32 (histograms).
__global__ void __launch_bounds__(256) select_kernel(const float *__restrict__ qt, const float *__restrict__ kt,
                                                     const int32_t *__restrict__ probe_list, const int64_t *__restrict__ row_ptr,
                                                     int32_t *__restrict__ col_idx, SelGeom g, HeadCfgArray cfg, int R) {
  const int h = blockIdx.y;
  const saf3r_head_cfg c = cfg.c[h];
  const int I0 = blockIdx.x * R;
  const int rows = (int)i64min(R, g.NB - I0);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  extern __shared__ float sm[];

  if (c.type != SAF3R_HEAD_BLOCK_TOPK) {
    for (int r = warp; r < rows; r += 8) {
      const int64_t I = I0 + r;
      int32_t *out = col_idx + row_ptr[(int64_t)h * g.NB + I];
      if (c.type == SAF3R_HEAD_QUERY_PROBE_TOPK) {
        const int n = (int)i64min(c.keep_blocks, g.NB);
        for (int i = lane; i < n; i += 32) out[i] = probe_list[(int64_t)h * g.NB + i];
      } else if (c.type == SAF3R_HEAD_DENSE) {
        for (int J = lane; J < g.NB; J += 32) out[J] = J;
      } else if (c.type == SAF3R_HEAD_UNIFORM_STRIDE && c.stride >= 1) {
        const int n = (g.NB - c.offset + c.stride - 1) / c.stride;
        for (int i = lane; i < n; i += 32) out[i] = c.offset + i * c.stride;
      } else if (lane == 0) {
        int64_t w = 0;
        closed_form_row(g, c, I, [&](int64_t J) { out[w++] = (int32_t)J; });
      }
    }
    return;
  }

  float *scores = sm;                                   // [R][NB]
  float *qrows = sm + (size_t)R * g.NB;                 // [R][64]
  uint32_t *hist = reinterpret_cast<uint32_t *>(qrows + R * 64) + warp * 256;
  for (int i = threadIdx.x; i < rows * 64; i += blockDim.x) qrows[i] = qt[((int64_t)h * g.NB + I0) * 64 + i];
  __syncthreads();
  const float cs = c.score_mode == SAF3R_SCORE_COSINE ? 1.f : 0.125f;
  for (int J = threadIdx.x; J < g.NB; J += blockDim.x) {
    float kv[64];
    const float4 *kr = reinterpret_cast<const float4 *>(kt + ((int64_t)h * g.NB + J) * 64);
#pragma unroll
    for (int d4 = 0; d4 < 16; ++d4) {
      const float4 t = __ldg(kr + d4);
      kv[4 * d4] = t.x; kv[4 * d4 + 1] = t.y; kv[4 * d4 + 2] = t.z; kv[4 * d4 + 3] = t.w;
    }
    for (int r = 0; r < rows; ++r) {
      const float4 *qr = reinterpret_cast<const float4 *>(qrows + r * 64);
      float acc = 0.f;
#pragma unroll
      for (int d4 = 0; d4 < 16; ++d4) {
        const float4 t = qr[d4];
        acc = fmaf(t.x, kv[4 * d4], acc);
        acc = fmaf(t.y, kv[4 * d4 + 1], acc);
        acc = fmaf(t.z, kv[4 * d4 + 2], acc);
        acc = fmaf(t.w, kv[4 * d4 + 3], acc);
      }
      scores[(size_t)r * g.NB + J] = acc * cs;
    }
  }
  __syncthreads();
  for (int r = warp; r < rows; r += 8) {
    int32_t *out = col_idx + row_ptr[(int64_t)h * g.NB + I0 + r];
    if (c.topk_scope == SAF3R_SCOPE_GLOBAL)
      warp_topn_emit(scores + (size_t)r * g.NB, g.NB, (int)i64min(c.keep_blocks, g.NB), out, hist);
    else
      warp_per_frame_emit(scores + (size_t)r * g.NB, g, c.topk_per_frame, out);
  }
}

}  // namespace saf3r
