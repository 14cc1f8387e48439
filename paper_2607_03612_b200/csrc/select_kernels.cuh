// Online pattern adaptation at block granularity (steps a-1..a-3 of DESIGN.md):
//   pool_rowptr_kernel  Q,K bf16 -> Qtilde,Ktilde fp32 block means (HBM-bound stream, one warp per block) and, in extra CTAs
//                       of the same launch, row_ptr from the closed-form row lengths
//   probe_kernel        qbar = (1/N) sum_t q_t from the pooled block means, p[J] = qbar . Ktilde_J / sqrt(D),
//                       top-n -> one shared list per QUERY_PROBE head
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

// ------------------------------------------------------------------------------------------------ pool + row_ptr
// One launch, two kinds of CTA (256 threads):
//   blockIdx.x <  pool_ctas : 8 warps, ONE WARP PER TOKEN BLOCK.  job j = (tensor, head) pairs that the head's rule reads
//                            (host-built list), warp w -> (job = w / NB, J = w % NB).  A warp streams its block's
//                            B x 128 B with 16-byte loads (lane = 16-byte chunk (l&7) of rows (l>>3) + 4i, eight loads in
//                            flight), accumulates in fp32, folds the four row groups with shuffles and writes the
//                            64-float mean.  No shared memory, no block barrier.
//   blockIdx.x >= pool_ctas : one CTA per head writes that head's row_ptr entries: head_base + I*len for heads whose
//                            rows all have the same length, a block scan of the closed-form lengths otherwise.
struct PoolJobs {
  int32_t n;                            // number of (tensor, head) jobs
  uint8_t head[2 * SAF3R_MAX_HEADS];
  uint8_t which[2 * SAF3R_MAX_HEADS];   // 0 = Q, 1 = K
  uint8_t cosine[2 * SAF3R_MAX_HEADS];  // L2-normalise each token first
  uint8_t part[2 * SAF3R_MAX_HEADS];    // also write per-CTA token sums (Q of a QUERY_PROBE head, for qbar)
};
struct RowPtrPlan {
  int64_t head_base[SAF3R_MAX_HEADS + 1];  // first entry of each head (host closed form); [H] = total
  int32_t const_len[SAF3R_MAX_HEADS];      // >= 0: every row of the head has this length; -1: per-row closed form
};

__device__ __forceinline__ uint4 ld_stream_16(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

__global__ void __launch_bounds__(256) pool_rowptr_kernel(const __nv_bfloat16 *__restrict__ q, const __nv_bfloat16 *__restrict__ k,
                                                          float *__restrict__ qt, float *__restrict__ ktT, float *__restrict__ qpart,
                                                          int64_t *__restrict__ row_ptr, SelGeom g, PoolJobs jobs, RowPtrPlan plan,
                                                          HeadCfgArray cfg, int pool_ctas) {
  if ((int)blockIdx.x >= pool_ctas) {
    // ---------------------------------------------------------------- row_ptr of one head
    const int h = blockIdx.x - pool_ctas;
    int64_t *rp = row_ptr + (int64_t)h * g.NB;
    const int64_t base = plan.head_base[h];
    if (plan.const_len[h] >= 0) {
      for (int I = threadIdx.x; I < g.NB; I += 256) rp[I] = base + (int64_t)I * plan.const_len[h];
    } else {
      __shared__ int64_t sums[256];
      const int per = (g.NB + 255) / 256;
      const int a = min(g.NB, (int)threadIdx.x * per), b = min(g.NB, a + per);
      int64_t s = 0;
      for (int I = a; I < b; ++I) s += row_length(g, cfg.c[h], I);
      sums[threadIdx.x] = s;
      __syncthreads();
      for (int off = 1; off < 256; off <<= 1) {
        int64_t v = (int)threadIdx.x >= off ? sums[threadIdx.x - off] : 0;
        __syncthreads();
        sums[threadIdx.x] += v;
        __syncthreads();
      }
      int64_t run = base + (threadIdx.x ? sums[threadIdx.x - 1] : 0);
      for (int I = a; I < b; ++I) {
        rp[I] = run;
        run += row_length(g, cfg.c[h], I);
      }
    }
    if (h == g.H - 1 && threadIdx.x == 0) row_ptr[(int64_t)g.H * g.NB] = plan.head_base[g.H];
    return;
  }
  // ------------------------------------------------------------------ pool: one warp per token block
  // CTA c of a job covers blocks 8c .. 8c+7 (jobs are padded to a multiple of 8 blocks, so a CTA never straddles jobs)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ctas_per_job = (g.NB + 7) / 8;
  const int job = blockIdx.x / ctas_per_job, cta_in_job = blockIdx.x % ctas_per_job;
  const int J = cta_in_job * 8 + warp;
  __shared__ float qsum[8][64];
  const bool want_part = jobs.part[job] != 0;  // Q of a QUERY_PROBE head: also emit this CTA's token sum (for qbar)
  if (J >= g.NB) {
    if (want_part) {
      qsum[warp][lane] = 0.f;
      qsum[warp][lane + 32] = 0.f;
      __syncthreads();
    }
    return;
  }
  const int h = jobs.head[job], which = jobs.which[job];
  const bool cosine = jobs.cosine[job] != 0;
  const int64_t t0 = (int64_t)J * g.B;
  const int cnt = (int)i64min(g.B, g.N - t0);
  const int sub = lane & 7, rg = lane >> 3;
  const __nv_bfloat16 *src = (which ? k : q) + (int64_t)h * g.stride_head + t0 * g.stride_token + sub * 8;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  for (int r0 = 0; r0 < g.B; r0 += 32) {  // 8 loads of 16 B in flight per lane (rows r0 + rg + 4i)
    uint4 raw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = r0 + rg + 4 * i;
      raw[i] = make_uint4(0, 0, 0, 0);
      if (r < cnt) raw[i] = ld_stream_16(src + (int64_t)r * g.stride_token);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const uint32_t w[4] = {raw[i].x, raw[i].y, raw[i].z, raw[i].w};
      float v[8];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        v[2 * c] = __uint_as_float(w[c] << 16);
        v[2 * c + 1] = __uint_as_float(w[c] & 0xFFFF0000u);
      }
      float inv = 1.f;
      if (cosine) {
        float ss = 0.f;
#pragma unroll
        for (int c = 0; c < 8; ++c) ss = fmaf(v[c], v[c], ss);
        ss += __shfl_xor_sync(0xffffffffu, ss, 1);
        ss += __shfl_xor_sync(0xffffffffu, ss, 2);
        ss += __shfl_xor_sync(0xffffffffu, ss, 4);
        const float nrm = sqrtf(ss);
        inv = nrm < 1e-20f ? 0.f : 1.f / nrm;
      }
#pragma unroll
      for (int c = 0; c < 8; ++c) acc[c] = fmaf(v[c], inv, acc[c]);
    }
  }
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], 8);
    acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], 16);
  }
  const float invc = 1.f / (float)cnt;
  if (rg == 0) {
    if (which == 0) {  // Qtilde row-major [H][NB][64]
      float4 *dst = reinterpret_cast<float4 *>(qt + ((int64_t)h * g.NB + J) * 64 + sub * 8);
      dst[0] = make_float4(acc[0] * invc, acc[1] * invc, acc[2] * invc, acc[3] * invc);
      dst[1] = make_float4(acc[4] * invc, acc[5] * invc, acc[6] * invc, acc[7] * invc);
    } else {  // Ktilde TRANSPOSED [H][64][NB]: the score kernels read it coalesced over J
#pragma unroll
      for (int c = 0; c < 8; ++c) ktT[((int64_t)h * 64 + sub * 8 + c) * g.NB + J] = acc[c] * invc;
    }
  }
  if (want_part) {
    if (rg == 0) {
#pragma unroll
      for (int c = 0; c < 8; ++c) qsum[warp][sub * 8 + c] = acc[c];
    }
    __syncthreads();
    if (warp == 0) {  // warp 0 always owns a real block (J = 8c < NB)
#pragma unroll
      for (int d = lane; d < 64; d += 32) {
        float t = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += qsum[w][d];
        qpart[((int64_t)h * ctas_per_job + cta_in_job) * 64 + d] = t;
      }
    }
  }
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
// grid (number of QUERY_PROBE heads), 1024 threads, dynamic smem: NB floats + 256 uint32.  qbar (16 row groups x 64 dims,
// fixed summation order), probe scores, then warp 0 radix-selects.  Writes the head's shared list to probe_list[h][0..n).
struct ProbeHeads { int32_t n; uint8_t head[SAF3R_MAX_HEADS]; };

__global__ void __launch_bounds__(1024) probe_kernel(const float *__restrict__ qpart, const float *__restrict__ ktT,
                                                     int32_t *__restrict__ probe_list, SelGeom g, HeadCfgArray cfg, ProbeHeads ph) {
  const int h = ph.head[blockIdx.x];
  extern __shared__ float sm[];
  float *s = sm;
  uint32_t *hist = reinterpret_cast<uint32_t *>(sm + g.NB);
  __shared__ float part[16][64];
  __shared__ float qb[64];
  {
    const int d = threadIdx.x & 63, grp = threadIdx.x >> 6;
    const int nparts = (g.NB + 7) / 8;
    const float *base = qpart + (int64_t)h * nparts * 64 + d;
    float a0 = 0.f;
    for (int c = grp; c < nparts; c += 16) a0 += base[(int64_t)c * 64];
    part[grp][d] = a0;
    __syncthreads();
    if (threadIdx.x < 64) {
      float t = 0.f;
#pragma unroll
      for (int i = 0; i < 16; ++i) t += part[i][threadIdx.x];
      qb[threadIdx.x] = t / (float)g.N;
    }
    __syncthreads();
  }
  for (int J = threadIdx.x; J < g.NB; J += blockDim.x) {
    const float *kc = ktT + (int64_t)h * 64 * g.NB + J;
    float acc = 0.f;
#pragma unroll 16
    for (int d = 0; d < 64; ++d) acc = fmaf(qb[d], __ldg(kc + (int64_t)d * g.NB), acc);
    s[J] = acc * 0.125f;
  }
  __syncthreads();
  if (threadIdx.x < 32) warp_topn_emit(s, g.NB, (int)i64min(cfg.c[h].keep_blocks, g.NB), probe_list + (int64_t)h * g.NB, hist);
}

// ------------------------------------------------------------------------------------------------ select
// grid (ceil(NB/R), H), 256 threads (8 warps), R <= 16 rows per CTA (Ktilde is re-read once per CTA, so more rows = less L2 traffic).  dynamic smem: R*NB floats (scores) + R*64 floats
// (Qtilde rows) + 8*256 uint32 (histograms).
__global__ void __launch_bounds__(256) select_kernel(const float *__restrict__ qt, const float *__restrict__ ktT,
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
      } else if (c.type == SAF3R_HEAD_UNIFORM_STRIDE) {  // keep_blocks form (n <= NB, so the indices are distinct)
        for (int i = lane; i < c.keep_blocks; i += 32) out[i] = (int32_t)(((int64_t)i * g.NB) / c.keep_blocks);
      } else if (c.type == SAF3R_HEAD_STATIC && c.static_mode != SAF3R_STATIC_POSITION_BAND) {  // one contiguous range
        int64_t lo, hi;
        if (c.static_mode == SAF3R_STATIC_ANCHOR) {
          lo = ((int64_t)c.anchor_frame * g.T) / g.B;
          hi = (((int64_t)c.anchor_frame + 1) * g.T - 1) / g.B;
        } else {
          const int64_t t0 = I * g.B, t1 = i64min(t0 + g.B, g.N);
          lo = ((t0 / g.T) * g.T) / g.B;
          hi = (((t1 - 1) / g.T + 1) * g.T - 1) / g.B;
        }
        for (int64_t J = lo + lane; J <= hi; J += 32) out[J - lo] = (int32_t)J;
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
    const float *kc = ktT + (int64_t)h * 64 * g.NB + J;
#pragma unroll
    for (int d = 0; d < 64; ++d) kv[d] = __ldg(kc + (int64_t)d * g.NB);
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
