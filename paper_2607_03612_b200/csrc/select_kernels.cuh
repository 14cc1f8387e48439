// Online pattern adaptation at block granularity (steps a-1..a-3 of DESIGN.md):
//   select_fused_kernel  ONE persistent launch; its CTAs draw tasks in a fixed order from a ticket counter:
//     pool tasks    Q,K bf16 -> Qtilde,Ktilde fp32 block means and per-task token sums of Q (the HBM-bound stream)
//     row_ptr tasks closed-form row lengths -> offsets
//     score strips  per (BLOCK_TOPK head, strip of q-blocks): score rows in shared memory + top-n / per-frame top-k
//     probe tasks   per QUERY_PROBE head: qbar = (1/N) sum_t q_t, p[J] = qbar . Ktilde_J / sqrt(D), top-n -> lists
//     light / emit  per-row closed forms, copies from the index cache, constant-length closed-form lists
//   the dependent tasks are interleaved with the pool tasks of the heads pooled later, so they run under the HBM stream
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

// Ktilde is stored TRANSPOSED, [H][64][NBp] with the row stride NBp = NB rounded up to 4, so that the score stage reads
// four consecutive k-blocks of one dimension d as one aligned 16-byte load, coalesced across the warp.
__host__ __device__ inline int64_t kt_stride(int32_t NB) { return ((int64_t)NB + 3) & ~(int64_t)3; }

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
  const bool topk = c.type == SAF3R_HEAD_BLOCK_TOPK || c.type == SAF3R_HEAD_CACHED;  // CACHED repeats its source head's rule
  if (c.type == SAF3R_HEAD_QUERY_PROBE_TOPK || (topk && c.topk_scope == SAF3R_SCOPE_GLOBAL))
    return i64min(c.keep_blocks, g.NB);
  if (topk) {
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

// ------------------------------------------------------------------------------------------------ warp-level top-n
// Order-preserving key: larger float <-> larger key; -0 is folded onto +0 so that ties follow the float comparison.
__device__ __forceinline__ uint32_t score_key(float s) {
  uint32_t u = __float_as_uint(s);
  if (u == 0x80000000u) u = 0u;
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// rows with NB <= 32*36 (or <= 32*72) keep their keys in registers during the bisection; longer rows re-read shared memory

// One warp: keep the n largest of key[0..NB) (order-preserving keys in shared memory) under (key desc, index asc);
// write their indices ascending to out.  No atomics, no sort: a bitwise bisection finds the n-th largest key tau (one
// warp-wide count of {key >= candidate} per bit, keys distributed over the lanes; it stops early as soon as a candidate
// splits the row into exactly n and NB-n keys), then an ordered ballot compaction emits {key > tau} plus the first
// `need` (by index) of {key == tau}.
template <int kKeysPerLaneReg>  // 0: keys stay in shared memory
__device__ __forceinline__ void warp_topn_bisect_impl(const uint32_t *key, int NB, int n, int32_t *out, int base) {
  constexpr bool kRegs = kKeysPerLaneReg > 0;
  const int lane = threadIdx.x & 31;
  uint32_t kk[kRegs ? kKeysPerLaneReg : 1];
  if (kRegs) {
#pragma unroll
    for (int i = 0; i < kKeysPerLaneReg; ++i) {
      const int j = lane + 32 * i;
      kk[i] = j < NB ? key[j] : 0u;  // key 0 is below every candidate (candidates have at least one bit set)
    }
  }
  auto count_ge = [&](uint32_t cand) -> int {
    int c0 = 0, c1 = 0;  // two chains; compare + predicated add = two instructions per key
    if (kRegs) {
#pragma unroll
      for (int i = 0; i < kKeysPerLaneReg; i += 2) {
        asm("{\n\t.reg .pred p;\n\tsetp.ge.u32 p, %1, %2;\n\t@p add.s32 %0, %0, 1;\n\t}" : "+r"(c0) : "r"(kk[i]), "r"(cand));
        asm("{\n\t.reg .pred p;\n\tsetp.ge.u32 p, %1, %2;\n\t@p add.s32 %0, %0, 1;\n\t}" : "+r"(c1) : "r"(kk[i + 1]), "r"(cand));
      }
    } else {
      for (int j = lane; j < NB; j += 32) c0 += (key[j] >= cand) ? 1 : 0;
    }
    return __reduce_add_sync(0xffffffffu, c0 + c1);
  };
  uint32_t prefix = 0;
  bool exact = false;
#pragma unroll 1
  for (int bit = 31; bit >= 0; --bit) {
    const uint32_t cand = prefix | (1u << bit);
    const int c = count_ge(cand);
    if (c >= n) {
      prefix = cand;
      if (c == n) { exact = true; break; }
    }
  }
  // exact: the kept set is {key >= prefix}, i.e. {key > prefix-1} with no ties to take.  Otherwise prefix is the n-th
  // largest key tau: keep {key > tau} and the first n - |{key > tau}| of the keys equal to tau.
  uint32_t tau;
  int need;
  if (exact) {
    tau = prefix - 1u;
    need = 0;
  } else {
    tau = prefix;
    need = n - (tau == 0xffffffffu ? 0 : count_ge(tau + 1u));
  }
  int written = 0, eq_seen = 0;
  const uint32_t lt = (1u << lane) - 1u;
  if (kRegs && need == 0) {  // common case: no ties at the cut; keys still in registers (padding keys are 0 <= tau)
#pragma unroll
    for (int i = 0; i < kKeysPerLaneReg; ++i) {
      const bool take = kk[i] > tau;
      const uint32_t tb = __ballot_sync(0xffffffffu, take);
      int32_t *dst = out + written + __popc(tb & lt);
      asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p st.global.u32 [%0], %1;\n\t}" ::"l"(dst), "r"(base + lane + 32 * i), "r"((uint32_t)take) : "memory");
      written += __popc(tb);
    }
    return;
  }
  for (int j0 = 0; j0 < NB; j0 += 32) {
    const int j = j0 + lane;
    const uint32_t kv = j < NB ? key[j] : 0u;
    const bool gt = j < NB && kv > tau, eq = j < NB && kv == tau && need > 0;
    const uint32_t eqb = __ballot_sync(0xffffffffu, eq);
    const bool take = gt || (eq && eq_seen + __popc(eqb & lt) < need);
    const uint32_t tb = __ballot_sync(0xffffffffu, take);
    if (take) out[written + __popc(tb & lt)] = base + j;
    written += __popc(tb);
    eq_seen += __popc(eqb);
  }
}
// `base` is added to every index written (the keys may be a window of a longer row)
// kSmall: the caller guarantees NB <= 32 * 36 (the three-CTAs-per-SM build of the fused kernel: 80 registers per thread)
template <bool kSmall = false>
__device__ __forceinline__ void warp_topn_bisect(const uint32_t *key, int NB, int n, int32_t *out, int base = 0) {
  if (kSmall || NB <= 32 * 36) warp_topn_bisect_impl<36>(key, NB, n, out, base);
  else if (NB <= 32 * 72) warp_topn_bisect_impl<72>(key, NB, n, out, base);
  else warp_topn_bisect_impl<0>(key, NB, n, out, base);
}

// One warp: per-frame top-k (PER_FRAME scope): in every frame's candidate range keep the kf best; ascending output.
__device__ inline void warp_per_frame_emit(const uint32_t *key, const SelGeom &g, int kf, int32_t *out) {
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
      const uint32_t sa = key[lo + a];
      int rank = 0;
      for (int b = 0; b < m; ++b) {
        const uint32_t sb = key[lo + b];
        rank += (sb > sa) || (sb == sa && b < a);
      }
      if (rank < kf) out[pos++] = (int32_t)(lo + a);
    }
    base += __shfl_sync(0xffffffffu, inc, 31);
  }
}

// ------------------------------------------------------------------------------------------------ light rows
// One warp writes the list of q-block I of a head whose rule needs no scores of its own: closed forms (DENSE,
// UNIFORM_STRIDE, STATIC) or a copy of the head's probe list (QUERY_PROBE_TOPK).
__device__ __forceinline__ void emit_light_row(const SelGeom &g, const saf3r_head_cfg &c, int h, int64_t I, int32_t *out,
                                               const int32_t *probe_list) {
  const int lane = threadIdx.x & 31;
  if (c.type == SAF3R_HEAD_QUERY_PROBE_TOPK) {
    const int n = (int)i64min(c.keep_blocks, g.NB);
    for (int i = lane; i < n; i += 32) out[i] = probe_list[(int64_t)h * g.NB + i];
  } else if (c.type == SAF3R_HEAD_DENSE) {
    for (int J = lane; J < g.NB; J += 32) out[J] = J;
  } else if (c.type == SAF3R_HEAD_UNIFORM_STRIDE && c.stride >= 1) {
    const int n = (g.NB - c.offset + c.stride - 1) / c.stride;
    for (int i = lane; i < n; i += 32) out[i] = c.offset + i * c.stride;
  } else if (c.type == SAF3R_HEAD_UNIFORM_STRIDE) {  // keep_blocks form (n <= NB, so the indices are distinct)
    if ((uint64_t)g.NB * (uint64_t)c.keep_blocks < 0x100000000ull) {  // 32-bit division (the 64-bit one is emulated)
      const uint32_t nb = (uint32_t)g.NB, kb = (uint32_t)c.keep_blocks;
      for (uint32_t i = lane; i < kb; i += 32) out[i] = (int32_t)((i * nb) / kb);
    } else {
      for (int i = lane; i < c.keep_blocks; i += 32) out[i] = (int32_t)(((int64_t)i * g.NB) / c.keep_blocks);
    }
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
  } else {
    // POSITION_BAND, lane-parallel: the row is a sequence of (frame, interval) block ranges [a_i, b_i]; b_i is a closed form and
    // a_i = max(first block of the interval, b_{i-1} + 1) only needs the previous range's END, so 32 ranges are sized at once
    // and placed with a warp prefix sum (same set and order as closed_form_row, which the host sizing uses)
    const int64_t T = g.T, B = g.B;
    const int64_t t0 = I * B, t1 = i64min(t0 + B, g.N);
    const int64_t f0 = t0 / T, f1 = (t1 - 1) / T, r = c.band_radius;
    int64_t lo[2], hi[2];
    int ni;
    if (f1 == f0) {
      lo[0] = i64max(0, t0 - f0 * T - r); hi[0] = i64min(T - 1, (t1 - 1) - f0 * T + r); ni = 1;
    } else if (f1 - f0 >= 2) {
      lo[0] = 0; hi[0] = T - 1; ni = 1;
    } else {
      const int64_t loA = i64max(0, t0 - f0 * T - r), hiB = i64min(T - 1, (t1 - 1) - f1 * T + r);
      if (hiB + 1 >= loA) { lo[0] = 0; hi[0] = T - 1; ni = 1; }
      else { lo[0] = 0; hi[0] = hiB; lo[1] = loA; hi[1] = T - 1; ni = 2; }
    }
    const int64_t items = (int64_t)g.S * ni;
    int64_t base = 0;
    for (int64_t i0 = 0; i0 < items; i0 += 32) {
      const int64_t i = i0 + lane;
      int64_t a = 0, b = -1;
      if (i < items) {
        const int64_t fr = i / ni;
        const int qi = (int)(i % ni);
        b = (fr * T + hi[qi]) / B;
        a = (fr * T + lo[qi]) / B;
        if (i > 0) {
          const int64_t pf = (i - 1) / ni;
          const int pq = (int)((i - 1) % ni);
          a = i64max(a, (pf * T + hi[pq]) / B + 1);  // the previous range's end (ends are non-decreasing)
        }
      }
      const int cnt = (int)i64max(0, b - a + 1);
      int inc = cnt;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += t;
      }
      int32_t *dst = out + base + inc - cnt;
      for (int j = 0; j < cnt; ++j) dst[j] = (int32_t)(a + j);
      base += __shfl_sync(0xffffffffu, inc, 31);
    }
  }
}
constexpr int kLightRows = 32;  // rows per CTA of the light emitters (8 warps x 4 rows)

// Which heads each kind of task serves (host-built).
struct HeadSets {
  int32_t n_emit, n_light, n_block, n_probe, n_cached;
  uint8_t cached[SAF3R_MAX_HEADS];  // CACHED heads (rows copied from the index cache; need row_ptr)
  uint8_t emit[SAF3R_MAX_HEADS];   // closed-form heads whose rows all have the same length (no dependence at all)
  uint8_t light[SAF3R_MAX_HEADS];  // per-row-length STATIC heads (need row_ptr)
  uint8_t block[SAF3R_MAX_HEADS];  // BLOCK_TOPK heads (score strips: scores + top-n)
  uint8_t probe[SAF3R_MAX_HEADS];  // QUERY_PROBE heads (probe-score chunks, one top-n task, list copies)
};

// ------------------------------------------------------------------------------------------------ pool / row_ptr / probe tasks
// (tasks of select_fused_kernel, each run by a whole 256-thread CTA; the ticket order is described at the kernel)
constexpr int kPoolBlocksPerTask = 8;  // one block per warp
constexpr int kPoolLoads = 16;         // independent 16-byte loads in flight per lane (64 token rows per round; 8 measured the same)
struct PoolJobs {
  int32_t n;                            // number of (tensor, head) jobs
  uint8_t head[2 * SAF3R_MAX_HEADS];
  uint8_t which[2 * SAF3R_MAX_HEADS];   // 0 = Q, 1 = K
  uint8_t cosine[2 * SAF3R_MAX_HEADS];  // L2-normalise each token first
  uint8_t probe[2 * SAF3R_MAX_HEADS];   // the head is a QUERY_PROBE head (its Q job also writes per-CTA token sums)
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

// Probe of a QUERY_PROBE head (qbar = (1/N) sum_t q_t, p[J] = qbar . Ktilde_J / sqrt(D)), as small tasks so that what
// is left to do after the head's last pool task is short and parallel:
//   probe_score_task  kProbeChunk k-blocks: qbar from the per-task token sums of the pool tasks (fixed order), the two halves of d by
//                     the two halves of the CTA (every load independent), keys -> probe_keys[h][J]
//   probe_topn_task   the head's NB keys -> shared memory, one warp runs the top-n -> probe_list[h][0..n)
constexpr int kProbeChunk = 128;
__device__ inline void probe_score_task(const float *qpart, const float *kt, uint32_t *probe_keys, const SelGeom &g, int h, int chunk,
                                        float (*part)[64], float *qb, float *ph /* [2][kProbeChunk] */) {
  const int nparts = (g.NB + kPoolBlocksPerTask - 1) / kPoolBlocksPerTask;
  {
    // 16 groups of 16 threads; a thread owns four dimensions and every 16th partial sum (independent 16-byte loads, eight in flight);
    // the groups are folded in a fixed order, so qbar does not depend on scheduling
    const int d4 = threadIdx.x & 15, grp = threadIdx.x >> 4;
    const float4 *base = reinterpret_cast<const float4 *>(qpart + (int64_t)h * nparts * 64) + d4;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int c0 = grp; c0 < nparts; c0 += 16 * 8) {
      float4 t[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) t[i] = (c0 + 16 * i < nparts) ? __ldcg(base + (int64_t)(c0 + 16 * i) * 16) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int i = 0; i < 8; ++i) { a.x += t[i].x; a.y += t[i].y; a.z += t[i].z; a.w += t[i].w; }
    }
    *reinterpret_cast<float4 *>(&part[grp][4 * d4]) = a;
    __syncthreads();
    if (threadIdx.x < 64) {
      float sum = 0.f;
#pragma unroll
      for (int gq = 0; gq < 16; ++gq) sum += part[gq][threadIdx.x];
      qb[threadIdx.x] = sum / (float)g.N;
    }
    __syncthreads();
  }
  const int64_t ld = kt_stride(g.NB);
  const int col = threadIdx.x & (kProbeChunk - 1), half = threadIdx.x / kProbeChunk;
  const int J = chunk * kProbeChunk + col;
  float acc = 0.f;
  if (J < g.NB) {
    const float *kc = kt + ((int64_t)h * 64 + 32 * half) * ld + J;
#pragma unroll
    for (int d0 = 0; d0 < 32; d0 += 16) {
      float t[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) t[i] = __ldcg(kc + (int64_t)(d0 + i) * ld);
#pragma unroll
      for (int i = 0; i < 16; ++i) acc = fmaf(qb[32 * half + d0 + i], t[i], acc);
    }
  }
  ph[half * kProbeChunk + col] = acc;
  __syncthreads();
  if (half == 0 && J < g.NB) probe_keys[(int64_t)h * g.NB + J] = score_key((ph[col] + ph[kProbeChunk + col]) * 0.125f);
}
template <bool kSmall>
__device__ inline void probe_topn_task(const uint32_t *probe_keys, int32_t *probe_list, const SelGeom &g, int h, int n,
                                       uint32_t *key /* dynamic smem, NB */) {
  for (int J = threadIdx.x; J < g.NB; J += 256) key[J] = __ldcg(probe_keys + (int64_t)h * g.NB + J);
  __syncthreads();
  if (threadIdx.x < 32) warp_topn_bisect<kSmall>(key, g.NB, n, probe_list + (int64_t)h * g.NB);
}

// row_ptr entries of head h (one task of the fused kernel, whole CTA)
__device__ inline void rowptr_task(int64_t *__restrict__ row_ptr, const SelGeom &g, const RowPtrPlan &plan, const HeadCfgArray &cfg, int h,
                                   int64_t *sums /* shared, 256 */) {
  int64_t *rp = row_ptr + (int64_t)h * g.NB;
  const int64_t base = plan.head_base[h];
  if (plan.const_len[h] >= 0) {
    for (int I = threadIdx.x; I < g.NB; I += 256) rp[I] = base + (int64_t)I * plan.const_len[h];
  } else {
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
}

// One pool task (whole CTA): eight consecutive token blocks of one (tensor, head) job, ONE WARP PER BLOCK and no shared memory on
// the way: a lane owns a 16-byte chunk (l & 7) of rows (l >> 3) + 4 i, kPoolLoads independent 16-byte loads in flight per lane and
// round of 4 * kPoolLoads rows, fp32 accumulate, optional per-token L2 normalisation (cosine), fold of the four row groups with shuffles,
// mean -> Qtilde (row-major) or Ktilde^T (transposed).  The Q job of a QUERY_PROBE head also leaves each warp's token sum in
// wsum for the task's partial sum of qbar, written by the caller after its barrier.
template <int kLoads>
__device__ __forceinline__ void pool_task(const __nv_bfloat16 *__restrict__ q, const __nv_bfloat16 *__restrict__ k, float *__restrict__ qt,
                                          float *__restrict__ kt, const SelGeom &g, const PoolJobs &jobs, int job, int task_in_job,
                                          float (*wsum)[64]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sub = lane & 7, rg = lane >> 3;
  const int J = task_in_job * kPoolBlocksPerTask + warp;
  const int h = jobs.head[job], which = jobs.which[job];
  const bool want_part = jobs.probe[job] != 0 && which == 0;
  const bool cosine = jobs.cosine[job] != 0;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (J < g.NB) {
    const int64_t t0 = (int64_t)J * g.B;
    const int cnt = (int)i64min(g.B, g.N - t0);
    const __nv_bfloat16 *src = (which ? k : q) + (int64_t)h * g.stride_head + t0 * g.stride_token + sub * 8;
#pragma unroll 1
    for (int r0 = 0; r0 < cnt; r0 += 4 * kLoads) {
      uint4 raw[kLoads];
#pragma unroll
      for (int i = 0; i < kLoads; ++i) {
        const int r = r0 + rg + 4 * i;
        raw[i] = make_uint4(0, 0, 0, 0);
        if (r < cnt) raw[i] = ld_stream_16(src + (int64_t)r * g.stride_token);
      }
#pragma unroll
      for (int i = 0; i < kLoads; ++i) {
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
    if (rg == 0) {
      if (which == 0) {
        float4 *dst = reinterpret_cast<float4 *>(qt + ((int64_t)h * g.NB + J) * 64 + sub * 8);  // Qtilde row-major [H][NB][64]
        dst[0] = make_float4(acc[0] / (float)cnt, acc[1] / (float)cnt, acc[2] / (float)cnt, acc[3] / (float)cnt);
        dst[1] = make_float4(acc[4] / (float)cnt, acc[5] / (float)cnt, acc[6] / (float)cnt, acc[7] / (float)cnt);
      } else {
        float *dst = kt + ((int64_t)h * 64 + sub * 8) * kt_stride(g.NB) + J;                    // Ktilde transposed [H][64][NBp]
#pragma unroll
        for (int c = 0; c < 8; ++c) dst[(int64_t)c * kt_stride(g.NB)] = acc[c] / (float)cnt;
      }
    }
  }
  if (want_part && rg == 0) {
#pragma unroll
    for (int c = 0; c < 8; ++c) wsum[warp][sub * 8 + c] = acc[c];  // zero for warps past the last block
  }
}

// ------------------------------------------------------------------------------------------------ score strips
// BLOCK_TOPK heads: score rows s[I][J] = Qtilde_I . Ktilde_J * c (fp32 FMA in the order d = 0..63, as packed row pairs) stored as
// order-preserving keys in shared memory (R rows x NB keys; the NB x NB matrix never exists), then one warp per row: bisection
// top-n or per-frame top-k.  Dynamic smem of a strip: R*NBp keys + 64*kSelRows floats (Qtilde rows, transposed so that four rows
// of one d are one 16-byte load) + the optional staging area of the left-over columns.
constexpr int kSelRows = 16;

__device__ __forceinline__ uint64_t sel_pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ uint64_t sel_fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}

// (Qtilde / Ktilde^T were written earlier in the SAME launch by other CTAs, so they are NOT read-only for this kernel: the
// read-only path (ld.global.nc / __ldg, or const __restrict__ letting the compiler pick it) is undefined for them under the PTX
// memory model.  They are read with ld.global.cg (__ldcg: L2 only, coherent) after the ld.acquire.gpu + bar.sync that follows the
// head's last pool task - the same loads probe_score_task uses.)
// Score rows I0 .. I0+rows-1 (rows <= RT) of head h against every k-block: keys[r][J] = key(Qtilde_{I0+r} . Ktilde_J * cs).
// Groups of 1024 columns: each thread owns four consecutive columns (one 16-byte load of Ktilde^T per d, coalesced across
// the warp) and RT rows, 4*RT accumulators as packed row pairs.  The columns left over (< 1024) are spread over all threads
// as (four rows, four columns) tasks.  Every sum runs in the order d = 0..63 with fp32 FMAs, so both paths give the same bits.
// When at most kSelTailCols columns are left over after the groups of 1024 (C3: NB = 1074 -> 52), their 64 x cols slice of
// Ktilde^T is copied to shared memory (kl) with cp.async while the groups are computed, and the tail becomes (row, column quad)
// tasks over all threads reading shared memory: one L2 round trip for the tail instead of a latency-bound pass of its own.
constexpr int kSelTailCols = 128;
template <int RT>
__device__ __forceinline__ void score_rows(const float *qt, const float *kt, uint32_t *keys, float *qT,
                                           const SelGeom &g, int h, int I0, int rows, float cs, float *kl) {
  for (int i = threadIdx.x; i < 64 * RT; i += blockDim.x) {
    const int d = i / RT, r = i % RT;
    qT[i] = r < rows ? __ldcg(qt + ((int64_t)h * g.NB + I0 + r) * 64 + d) : 0.f;
  }
  const int64_t ld = kt_stride(g.NB);
  const float *kh = kt + (int64_t)h * 64 * ld;
  const int Jtail = (g.NB / 1024) * 1024, tail_quads = (int)((ld - Jtail) / 4);
  const bool staged = kl != nullptr && Jtail > 0 && tail_quads * 4 <= kSelTailCols;
  if (staged) {
    for (int i = threadIdx.x; i < 64 * tail_quads; i += blockDim.x) {
      const int d = i / tail_quads, qd = i % tail_quads;
      const uint32_t dst = (uint32_t)__cvta_generic_to_shared(kl + (d * tail_quads + qd) * 4);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(kh + (int64_t)d * ld + Jtail + 4 * qd) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  __syncthreads();
  int Jb = 0;
  for (; Jb + 1024 <= g.NB; Jb += 1024) {
    const int J = Jb + 4 * (int)threadIdx.x;
    uint64_t a[4][RT / 2];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int r = 0; r < RT / 2; ++r) a[c][r] = 0ull;
    const float *kp = kh + J;
    constexpr int KB = RT <= 4 ? 16 : (RT <= 8 ? 8 : 4);  // 16-byte loads in flight per thread (short strips have the registers)
#pragma unroll 1
    for (int d0 = 0; d0 < 64; d0 += KB) {
      float4 kvb[KB];
#pragma unroll
      for (int i = 0; i < KB; ++i) kvb[i] = __ldcg(reinterpret_cast<const float4 *>(kp + (int64_t)(d0 + i) * ld));
#pragma unroll
      for (int i = 0; i < KB; ++i) {
        const float4 kv = kvb[i];
        const uint64_t k0 = sel_pack2(kv.x, kv.x), k1 = sel_pack2(kv.y, kv.y), k2 = sel_pack2(kv.z, kv.z), k3 = sel_pack2(kv.w, kv.w);
        const float4 *qr = reinterpret_cast<const float4 *>(qT + (d0 + i) * RT);
#pragma unroll
        for (int r4 = 0; r4 < RT / 4; ++r4) {
          const float4 t = qr[r4];
          const uint64_t qa = sel_pack2(t.x, t.y), qb = sel_pack2(t.z, t.w);
          a[0][2 * r4] = sel_fma2(qa, k0, a[0][2 * r4]);
          a[0][2 * r4 + 1] = sel_fma2(qb, k0, a[0][2 * r4 + 1]);
          a[1][2 * r4] = sel_fma2(qa, k1, a[1][2 * r4]);
          a[1][2 * r4 + 1] = sel_fma2(qb, k1, a[1][2 * r4 + 1]);
          a[2][2 * r4] = sel_fma2(qa, k2, a[2][2 * r4]);
          a[2][2 * r4 + 1] = sel_fma2(qb, k2, a[2][2 * r4 + 1]);
          a[3][2 * r4] = sel_fma2(qa, k3, a[3][2 * r4]);
          a[3][2 * r4 + 1] = sel_fma2(qb, k3, a[3][2 * r4 + 1]);
        }
      }
    }
#pragma unroll
    for (int r2 = 0; r2 < RT / 2; ++r2) {
      float lo[4], hi[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) asm("mov.b64 {%0, %1}, %2;" : "=f"(lo[c]), "=f"(hi[c]) : "l"(a[c][r2]));
      if (2 * r2 < rows)
        *reinterpret_cast<uint4 *>(keys + (size_t)(2 * r2) * ld + J) =
            make_uint4(score_key(lo[0] * cs), score_key(lo[1] * cs), score_key(lo[2] * cs), score_key(lo[3] * cs));
      if (2 * r2 + 1 < rows)
        *reinterpret_cast<uint4 *>(keys + (size_t)(2 * r2 + 1) * ld + J) =
            make_uint4(score_key(hi[0] * cs), score_key(hi[1] * cs), score_key(hi[2] * cs), score_key(hi[3] * cs));
    }
  }
  if (staged) {
    // (row, column quad) tasks from shared memory; the same fp32 FMA chain d = 0..63 as the packed form above, so the same bits
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    for (int idx = threadIdx.x; idx < rows * tail_quads; idx += blockDim.x) {
      const int r = idx / tail_quads, qd = idx % tail_quads;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll 16
      for (int d = 0; d < 64; ++d) {
        const float4 kv = *reinterpret_cast<const float4 *>(kl + (d * tail_quads + qd) * 4);
        const float qv = qT[d * RT + r];
        a0 = fmaf(qv, kv.x, a0); a1 = fmaf(qv, kv.y, a1); a2 = fmaf(qv, kv.z, a2); a3 = fmaf(qv, kv.w, a3);
      }
      *reinterpret_cast<uint4 *>(keys + (size_t)r * ld + Jtail + 4 * qd) =
          make_uint4(score_key(a0 * cs), score_key(a1 * cs), score_key(a2 * cs), score_key(a3 * cs));
    }
    return;
  }
  // left-over columns: (four rows, column quad) tasks; the padded columns NB..NBp-1 of Ktilde^T are never written, so their
  // scores are computed from garbage and stored into the row's padding, which nothing reads
  const int quads = (int)((ld - Jb) / 4);
  constexpr int RG = RT / 4;  // row groups of four
  for (int idx = threadIdx.x; idx < quads * RG; idx += blockDim.x) {
    const int rgp = idx / quads, J = Jb + 4 * (idx % quads);
    const float *kp = kh + J;
    uint64_t a[4][2];
#pragma unroll
    for (int c = 0; c < 4; ++c) a[c][0] = a[c][1] = 0ull;
#pragma unroll 8
    for (int d = 0; d < 64; ++d) {
      const float4 kv = __ldcg(reinterpret_cast<const float4 *>(kp + (int64_t)d * ld));
      const float4 t = *reinterpret_cast<const float4 *>(qT + d * RT + 4 * rgp);
      const uint64_t qa = sel_pack2(t.x, t.y), qb = sel_pack2(t.z, t.w);
      const uint64_t k0 = sel_pack2(kv.x, kv.x), k1 = sel_pack2(kv.y, kv.y), k2 = sel_pack2(kv.z, kv.z), k3 = sel_pack2(kv.w, kv.w);
      a[0][0] = sel_fma2(qa, k0, a[0][0]); a[0][1] = sel_fma2(qb, k0, a[0][1]);
      a[1][0] = sel_fma2(qa, k1, a[1][0]); a[1][1] = sel_fma2(qb, k1, a[1][1]);
      a[2][0] = sel_fma2(qa, k2, a[2][0]); a[2][1] = sel_fma2(qb, k2, a[2][1]);
      a[3][0] = sel_fma2(qa, k3, a[3][0]); a[3][1] = sel_fma2(qb, k3, a[3][1]);
    }
#pragma unroll
    for (int r2 = 0; r2 < 2; ++r2) {
      float lo[4], hi[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) asm("mov.b64 {%0, %1}, %2;" : "=f"(lo[c]), "=f"(hi[c]) : "l"(a[c][r2]));
      const int r = 4 * rgp + 2 * r2;
      if (r < rows)
        *reinterpret_cast<uint4 *>(keys + (size_t)r * ld + J) =
            make_uint4(score_key(lo[0] * cs), score_key(lo[1] * cs), score_key(lo[2] * cs), score_key(lo[3] * cs));
      if (r + 1 < rows)
        *reinterpret_cast<uint4 *>(keys + (size_t)(r + 1) * ld + J) =
            make_uint4(score_key(hi[0] * cs), score_key(hi[1] * cs), score_key(hi[2] * cs), score_key(hi[3] * cs));
    }
  }
}

// ------------------------------------------------------------------------------------------------ the fused selection kernel
// ONE persistent launch for the whole of saf3r_select.  CTAs (256 threads, <= 2 per SM) draw tickets from a device counter; the
// ticket order is a host-side closed form of (shape, cfg):
//   [row_ptr task per head] [pool tasks of the BLOCK_TOPK heads] [MIX: pool tasks of the QUERY_PROBE heads with one score strip
//   after every `period` of them] [what is left of either] [probe-score chunks] [probe top-n tasks] [light chunks] [emit chunks]
//   [probe-list copies]
// score strip: R q-block rows of a BLOCK_TOPK head (scores in shared memory, top-n / per-frame top-k); probe-score chunk: qbar and
// 128 entries of the probe row of a QUERY_PROBE head; probe top-n: one per QUERY_PROBE head (the row's top-n -> the head's list); light chunk: 32 rows of a per-row STATIC rule or of a CACHED head;
// emit chunk: 32 rows of a constant-length closed-form list; copy chunk: 32 of the NB identical rows of a QUERY_PROBE head.  So the score + select work of the BLOCK_TOPK heads and every list
// write run UNDER the HBM stream of the remaining pooling instead of after it, and nothing is launched twice.
// A task that needs the pooled tensors of head h spins (one thread, ld.acquire) on pooled[h]; every pool task ends with a
// release increment of it.  All tasks a waiter depends on have SMALLER tickets, i.e. were drawn by CTAs that are running and never
// wait on larger tickets: no deadlock whatever the grid size.  Light / CACHED tasks wait the same way for the head's row_ptr.
struct FusedPlan {
  int32_t t_begin, t_end;                 // tickets this launch serves (two launches when the stages are timed separately)
  int32_t n_rowptr, n_pool_a, n_pool_b;   // tasks per segment
  int32_t n_x, period;                    // score strips (mixed into the pool-B tasks, one after every `period` of them, >= 1)
  int32_t n_pscore, n_probe, n_light, n_emit, n_rep;  // after ALL pool tasks: probe-score chunks, probe top-n, light, emit, list copies
  int32_t pchunks;                        // probe-score chunks per QUERY_PROBE head
  int32_t strips, R, light_chunks;
  int32_t pool_need;                      // pool tasks per head = 2 jobs * tasks_per_job
  int32_t counter;                        // which ticket counter (0 / 1)
  int32_t tail_stage;                     // the strips have a shared-memory staging area for the left-over columns (score_rows)
};
constexpr int kSelScratch = 17 * 64 * 4 + 2 * kProbeChunk * 4;  // bytes of scratch of a probe-score task (partial sums of qbar, qbar, half sums)
constexpr int kSelCounters = 2 + 4 * SAF3R_MAX_HEADS;  // int32: 2 ticket counters, pooled[h], rowptr_done[h], probe_done[h], pscore_done[h]

__device__ __forceinline__ void wait_count(const int *ctr, int need) {
  if (threadIdx.x == 0) {
    int v;
    do {
      asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if (v < need) __nanosleep(200);
    } while (v < need);
  }
  __syncthreads();
}
__device__ __forceinline__ void signal_count(int *ctr) {
  __syncthreads();  // all threads of the CTA have issued their stores
  if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(ctr) : "memory");  // release: cumulative over the barrier
}

template <int kOcc>  // CTAs per SM the register budget is sized for (3: only strips of <= 8 rows and rows of <= 1152 keys)
__global__ void __launch_bounds__(256, kOcc) select_fused_kernel(const __nv_bfloat16 *__restrict__ q, const __nv_bfloat16 *__restrict__ k,
                                                              float *__restrict__ qt, float *__restrict__ kt, float *__restrict__ qpart,
                                                              uint32_t *__restrict__ probe_keys, int32_t *__restrict__ probe_list, int64_t *__restrict__ row_ptr,
                                                              int32_t *__restrict__ col_idx, const int64_t *__restrict__ cache_row_ptr,
                                                              const int32_t *__restrict__ cache_col_idx, int *__restrict__ counters,
                                                              SelGeom g, PoolJobs jobs, RowPtrPlan plan, HeadCfgArray cfg, HeadSets sets,
                                                              FusedPlan fp) {
  extern __shared__ __align__(16) float sm[];  // per task: score keys + Qtilde^T | probe keys | the scratch below (>= kSelScratch bytes)
  float(*wsum)[64] = reinterpret_cast<float(*)[64]>(sm);      // pool task: [8][64]
  int64_t *sums = reinterpret_cast<int64_t *>(sm);             // row_ptr task: [256]
  __shared__ int s_ticket;
  int *pooled = counters + 2, *rp_done = counters + 2 + SAF3R_MAX_HEADS, *probe_done = counters + 2 + 2 * SAF3R_MAX_HEADS,
      *pscore_done = counters + 2 + 3 * SAF3R_MAX_HEADS;
  const int warp = threadIdx.x >> 5;
  // thread 0 always holds the NEXT ticket: its atomic is issued a whole task ahead, so its latency never shows
  int next = 0;
  if (threadIdx.x == 0) next = fp.t_begin + atomicAdd(counters + fp.counter, 1);
  for (;;) {
    __syncthreads();  // the previous task is finished with the shared buffers (and with s_ticket)
    if (threadIdx.x == 0) s_ticket = next;
    __syncthreads();
    int t = s_ticket;
    if (t >= fp.t_end) break;
    if (threadIdx.x == 0) next = fp.t_begin + atomicAdd(counters + fp.counter, 1);
    // ---------------------------------------------------------------- decode the ticket
    int pool_task_id = -1, x = -1;
    if (t < fp.n_rowptr) {
      rowptr_task(row_ptr, g, plan, cfg, t, sums);
      signal_count(rp_done + t);
      continue;
    }
    t -= fp.n_rowptr;
    if (t < fp.n_pool_a) {
      pool_task_id = t;
    } else {
      t -= fp.n_pool_a;
      const int groups = min(fp.n_x, fp.n_pool_b / fp.period);  // full (period pool tasks, one dependent task) groups
      const int mixed = groups * (fp.period + 1);
      if (t < mixed) {
        const int gi = t / (fp.period + 1), r = t % (fp.period + 1);
        if (r < fp.period) pool_task_id = fp.n_pool_a + gi * fp.period + r;
        else x = gi;
      } else {
        t -= mixed;
        const int rest_pool = fp.n_pool_b - groups * fp.period;
        if (t < rest_pool) pool_task_id = fp.n_pool_a + groups * fp.period + t;
        else x = groups + (t - rest_pool);  // past n_x: the probe tasks
      }
    }
    if (pool_task_id >= 0) {
      const int tasks_per_job = (g.NB + kPoolBlocksPerTask - 1) / kPoolBlocksPerTask;
      const int job = pool_task_id / tasks_per_job, task_in_job = pool_task_id % tasks_per_job;
      pool_task<(kOcc > 2 ? 8 : kPoolLoads)>(q, k, qt, kt, g, jobs, job, task_in_job, wsum);
      if (jobs.probe[job] != 0 && jobs.which[job] == 0) {  // the task's token sum for qbar, warps in a fixed order
        __syncthreads();
        if (threadIdx.x < 64) {
          float tsum = 0.f;
#pragma unroll
          for (int w = 0; w < 8; ++w) tsum += wsum[w][threadIdx.x];
          qpart[((int64_t)jobs.head[job] * tasks_per_job + task_in_job) * 64 + threadIdx.x] = tsum;
        }
      }
      signal_count(pooled + jobs.head[job]);
      continue;
    }
    // ---------------------------------------------------------------- dependent tasks
    if (x < fp.n_x) {
      const int h = sets.block[x / fp.strips];
      const saf3r_head_cfg c = cfg.c[h];
      const int R = fp.R, I0 = (x % fp.strips) * R;
      const int rows = (int)i64min(R, g.NB - I0);
      wait_count(pooled + h, fp.pool_need);
      uint32_t *keys = reinterpret_cast<uint32_t *>(sm);   // [R][NBp]
      const int64_t ld = kt_stride(g.NB);
      float *qT = sm + (size_t)R * ld;                     // [64][RT] (rows past `rows` are zero)
      const float cs = c.score_mode == SAF3R_SCORE_COSINE ? 1.f : 0.125f;
      float *kl = fp.tail_stage ? qT + 64 * kSelRows : nullptr;  // [64][tail quads][4] staging of the left-over columns
      if (R <= 4) score_rows<4>(qt, kt, keys, qT, g, h, I0, rows, cs, kl);
      else if (R <= 8) score_rows<8>(qt, kt, keys, qT, g, h, I0, rows, cs, kl);
      else if constexpr (kOcc <= 2) score_rows<kSelRows>(qt, kt, keys, qT, g, h, I0, rows, cs, kl);
      __syncthreads();
      const int64_t base = plan.head_base[h];  // BLOCK_TOPK rows all have the same length: offsets are a closed form
      const int len = plan.const_len[h];
      for (int r = warp; r < rows; r += 8) {
        int32_t *out = col_idx + base + (int64_t)(I0 + r) * len;
        if (c.topk_scope == SAF3R_SCOPE_GLOBAL) warp_topn_bisect<(kOcc > 2)>(keys + (size_t)r * ld, g.NB, (int)i64min(c.keep_blocks, g.NB), out);
        else warp_per_frame_emit(keys + (size_t)r * ld, g, c.topk_per_frame, out);
      }
      continue;
    }
    x -= fp.n_x;
    if (x < fp.n_pscore) {
      const int h = sets.probe[x / fp.pchunks];
      wait_count(pooled + h, fp.pool_need);
      float(*part)[64] = reinterpret_cast<float(*)[64]>(sm);  // [16][64], then qbar [64], then the half sums [2][kProbeChunk]
      probe_score_task(qpart, kt, probe_keys, g, h, x % fp.pchunks, part, sm + 16 * 64, sm + 17 * 64);
      signal_count(pscore_done + h);
      continue;
    }
    x -= fp.n_pscore;
    if (x < fp.n_probe) {
      const int h = sets.probe[x];
      wait_count(pscore_done + h, fp.pchunks);
      probe_topn_task<(kOcc > 2)>(probe_keys, probe_list, g, h, (int)i64min(cfg.c[h].keep_blocks, g.NB), reinterpret_cast<uint32_t *>(sm));
      signal_count(probe_done + h);
      continue;
    }
    x -= fp.n_probe;
    if (x < fp.n_light) {
      const int I0 = (x % fp.light_chunks) * kLightRows, hi = x / fp.light_chunks;
      if (hi >= sets.n_light) {  // CACHED head: rows copied from the index cache
        const int h = sets.cached[hi - sets.n_light];
        wait_count(rp_done + h, 1);
        const int src = cfg.c[h].offset, lane = threadIdx.x & 31;
        for (int r = warp; r < kLightRows && I0 + r < g.NB; r += 8) {
          const int64_t a = cache_row_ptr[(int64_t)src * g.NB + I0 + r], b = cache_row_ptr[(int64_t)src * g.NB + I0 + r + 1];
          const int64_t o = row_ptr[(int64_t)h * g.NB + I0 + r], cap = row_ptr[(int64_t)h * g.NB + I0 + r + 1] - o;
          const int64_t n = i64min(b - a, cap);  // equal when cfg repeats the source rule; never write past the row
          for (int64_t i = lane; i < n; i += 32) col_idx[o + i] = cache_col_idx[a + i];
        }
      } else {
        const int h = sets.light[hi];
        wait_count(rp_done + h, 1);
        for (int r = warp; r < kLightRows && I0 + r < g.NB; r += 8)
          emit_light_row(g, cfg.c[h], h, I0 + r, col_idx + row_ptr[(int64_t)h * g.NB + I0 + r], nullptr);
      }
      continue;
    }
    x -= fp.n_light;
    if (x < fp.n_emit) {  // constant-length closed-form head: no dependence at all
      const int h = sets.emit[x / fp.light_chunks];
      const int I0 = (x % fp.light_chunks) * kLightRows;
      for (int r = warp; r < kLightRows && I0 + r < g.NB; r += 8)
        emit_light_row(g, cfg.c[h], h, I0 + r, col_idx + plan.head_base[h] + (int64_t)(I0 + r) * plan.const_len[h], nullptr);
      continue;
    }
    x -= fp.n_emit;
    {  // 32 of the NB identical rows of a QUERY_PROBE head: the region is the head's list repeated, written with coalesced stores
      const int h = sets.probe[x / fp.light_chunks];
      const int I0 = (x % fp.light_chunks) * kLightRows;
      const int n = (int)i64min(cfg.c[h].keep_blocks, g.NB);
      wait_count(probe_done + h, 1);
      int32_t *list = reinterpret_cast<int32_t *>(sm);
      for (int i = threadIdx.x; i < n; i += 256) list[i] = __ldcg(probe_list + (int64_t)h * g.NB + i);
      __syncthreads();
      const int nrows = min(kLightRows, g.NB - I0);
      int32_t *dst = col_idx + plan.head_base[h] + (int64_t)I0 * n;
      const int64_t total = (int64_t)nrows * n;
      int m = (int)(((int64_t)threadIdx.x) % n);
      const int step = 256 % n;
      for (int64_t idx = threadIdx.x; idx < total; idx += 256) {
        dst[idx] = list[m];
        m += step;
        if (m >= n) m -= n;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ list validation
// grid-stride over the H*NB rows: row_ptr non-decreasing, every row ascending, unique and inside [0, NB).  Counts bad rows.
__global__ void __launch_bounds__(256) check_lists_kernel(const int64_t *__restrict__ row_ptr, const int32_t *__restrict__ col_idx,
                                                          int64_t rows, int32_t NB, int64_t capacity, unsigned long long *bad) {
  for (int64_t r = (int64_t)blockIdx.x * 256 + threadIdx.x; r < rows; r += (int64_t)gridDim.x * 256) {
    const int64_t a = row_ptr[r], b = row_ptr[r + 1];
    bool ok = a >= 0 && b >= a && b <= capacity && b - a <= NB;
    if (ok) {
      int32_t prev = -1;
      for (int64_t i = a; i < b; ++i) {
        const int32_t J = col_idx[i];
        ok = ok && J > prev && J < NB;
        prev = J;
      }
    }
    if (!ok) atomicAdd(bad, 1ull);
  }
}

// ------------------------------------------------------------------------------------------------ list union (NEXT-4)
// out(h, I) = list_a(h, I) U list_b(h, I), ascending and unique ("combining Top-K with uniform striding").  Both
// inputs are ascending and unique, so one thread walks a row of each with two cursors.  Three launches: count (row lengths into
// out_row_ptr[r + 1]), an in-place inclusive scan by one CTA, write.  Entries past `capacity` are not written; the total in
// out_row_ptr[rows] tells the caller.
template <bool kWrite>
__global__ void __launch_bounds__(128) union_rows_kernel(const int64_t *__restrict__ rp_a, const int32_t *__restrict__ col_a,
                                                         const int64_t *__restrict__ rp_b, const int32_t *__restrict__ col_b,
                                                         int64_t *__restrict__ rp_o, int32_t *__restrict__ col_o, int64_t rows,
                                                         int64_t capacity) {
  const int64_t r = (int64_t)blockIdx.x * 128 + threadIdx.x;
  if (r >= rows) return;
  int64_t a = rp_a[r], b = rp_b[r];
  const int64_t a1 = rp_a[r + 1], b1 = rp_b[r + 1];
  int64_t o = kWrite ? rp_o[r] : 0;
  int32_t ja = a < a1 ? col_a[a] : INT32_MAX, jb = b < b1 ? col_b[b] : INT32_MAX;
  while (a < a1 || b < b1) {
    const int32_t j = ja < jb ? ja : jb;
    if (kWrite && o < capacity) col_o[o] = j;
    ++o;
    if (ja == j) { ++a; ja = a < a1 ? col_a[a] : INT32_MAX; }
    if (jb == j) { ++b; jb = b < b1 ? col_b[b] : INT32_MAX; }
  }
  if (!kWrite) rp_o[r + 1] = o;
}

// rp[0] = 0 and rp[1..rows] hold row lengths: turn them into offsets (inclusive scan in place), one CTA of 1024 threads.
__global__ void __launch_bounds__(1024) scan_row_ptr_kernel(int64_t *__restrict__ rp, int64_t rows) {
  __shared__ int64_t part[1024];
  const int64_t per = (rows + 1023) / 1024;
  const int64_t a = threadIdx.x * per < rows ? threadIdx.x * per : rows, b = a + per < rows ? a + per : rows;
  int64_t s = 0;
  for (int64_t i = a; i < b; ++i) s += rp[i + 1];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    const int64_t v = (int)threadIdx.x >= off ? part[threadIdx.x - off] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  int64_t run = threadIdx.x ? part[threadIdx.x - 1] : 0;
  if (threadIdx.x == 0) rp[0] = 0;
  for (int64_t i = a; i < b; ++i) {
    run += rp[i + 1];
    rp[i + 1] = run;
  }
}

}  // namespace saf3r
