// Token-granular variants: the paper's own token-level definitions of two of its kernels.
//   Uniform Sampling Kernel: every s-th key token -> no kernel of its own: a strided TMA view of K/V fed to the
//       dense mode of saf3r_attn_kernel (saf3r_token_stride_attn in saf3r_api.cu).
//   Query-Probe Top-K Kernel: qbar = (1/N) sum_i q_i, p[j] = qbar . k_j / sqrt(D) for every key TOKEN,
//       top-K tokens shared by all queries:
//         token_qsum_kernel    per-chunk token sums of Q (HBM stream)
//         token_probe_kernel   qbar from the chunk sums (fixed order), p[j] as order-preserving keys (HBM stream of K)
//         token_topk_kernel    one CTA per head: 11+11+10-bit radix select of the K-th largest key over N keys (first digit's
//                              histogram from the probe pass), then an ordered block compaction -> ascending indices, ties by lower index
//         token_gather_kernel  K/V rows of the selected tokens -> compact [H][K][64] tiles for the dense mode of the attention
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"
#include "select_kernels.cuh"

namespace saf3r {

constexpr int kTokChunk = 2048;  // tokens per CTA of the Q-sum pass
constexpr int kTokTile = 1024;   // tokens per CTA of the probe pass

__device__ __forceinline__ void bf16x8_to_f32(const uint4 &raw, float (&v)[8]) {
  const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    v[2 * c] = __uint_as_float(w[c] << 16);
    v[2 * c + 1] = __uint_as_float(w[c] & 0xFFFF0000u);
  }
}

// grid (ceil(N / kTokChunk), H), 256 threads: lane group of 8 threads = one token row (16 B each), 32 rows per step.
constexpr int kTokBins1 = 2048;  // histogram of the top 11 key bits, built by the probe pass for the top-K pass

__global__ void __launch_bounds__(256) token_qsum_kernel(const __nv_bfloat16 *__restrict__ q, float *__restrict__ part,
                                                         uint32_t *__restrict__ hist1, SelGeom g) {
  const int h = blockIdx.y, chunk = blockIdx.x;
  if (chunk == 0)  // the probe launch that follows accumulates into it
    for (int i = threadIdx.x; i < kTokBins1; i += 256) hist1[(int64_t)h * kTokBins1 + i] = 0u;
  const int sub = threadIdx.x & 7, row = threadIdx.x >> 3;
  const int64_t t0 = (int64_t)chunk * kTokChunk;
  const int cnt = (int)i64min(kTokChunk, g.N - t0);
  const __nv_bfloat16 *src = q + (int64_t)h * g.stride_head + t0 * g.stride_token + sub * 8;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  for (int r0 = 0; r0 < kTokChunk; r0 += 32 * 8) {
    uint4 raw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = r0 + row + 32 * i;
      raw[i] = make_uint4(0, 0, 0, 0);
      if (r < cnt) raw[i] = ld_stream_16(src + (int64_t)r * g.stride_token);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float v[8];
      bf16x8_to_f32(raw[i], v);
#pragma unroll
      for (int c = 0; c < 8; ++c) acc[c] += v[c];
    }
  }
  __shared__ float red[32][64];
#pragma unroll
  for (int c = 0; c < 8; ++c) red[row][sub * 8 + c] = acc[c];
  __syncthreads();
  if (threadIdx.x < 64) {
    float t = 0.f;
#pragma unroll
    for (int r = 0; r < 32; ++r) t += red[r][threadIdx.x];
    part[((int64_t)h * gridDim.x + chunk) * 64 + threadIdx.x] = t;
  }
}

// grid (ceil(N / kTokTile), H), 256 threads.  keys[h][j] = order-preserving key of p[j] = qbar . k_j / sqrt(D).
__global__ void __launch_bounds__(256) token_probe_kernel(const __nv_bfloat16 *__restrict__ k, const float *__restrict__ part,
                                                          uint32_t *__restrict__ keys, uint32_t *__restrict__ hist1, SelGeom g,
                                                          int n_chunks) {
  const int h = blockIdx.y;
  __shared__ float qb[64];
  __shared__ uint32_t sh1[kTokBins1];
  for (int i = threadIdx.x; i < kTokBins1; i += 256) sh1[i] = 0u;
  if (threadIdx.x < 64) {
    float t = 0.f;
    for (int c = 0; c < n_chunks; ++c) t += part[((int64_t)h * n_chunks + c) * 64 + threadIdx.x];  // fixed order
    qb[threadIdx.x] = t / (float)g.N;
  }
  __syncthreads();
  const int sub = threadIdx.x & 7, row = threadIdx.x >> 3;
  float qv[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) qv[c] = qb[sub * 8 + c];
  const int64_t t0 = (int64_t)blockIdx.x * kTokTile;
  const int cnt = (int)i64min(kTokTile, g.N - t0);
  const __nv_bfloat16 *src = k + (int64_t)h * g.stride_head + t0 * g.stride_token + sub * 8;
  for (int r0 = 0; r0 < kTokTile; r0 += 32 * 8) {
    uint4 raw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = r0 + row + 32 * i;
      raw[i] = make_uint4(0, 0, 0, 0);
      if (r < cnt) raw[i] = ld_stream_16(src + (int64_t)r * g.stride_token);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float v[8];
      bf16x8_to_f32(raw[i], v);
      float d = 0.f;
#pragma unroll
      for (int c = 0; c < 8; ++c) d = fmaf(qv[c], v[c], d);
      d += __shfl_xor_sync(0xffffffffu, d, 1);
      d += __shfl_xor_sync(0xffffffffu, d, 2);
      d += __shfl_xor_sync(0xffffffffu, d, 4);
      const int r = r0 + row + 32 * i;
      if (sub == 0 && r < cnt) {
        const uint32_t key = score_key(d * 0.125f);
        keys[(int64_t)h * g.N + t0 + r] = key;
        atomicAdd(&sh1[key >> 21], 1u);
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kTokBins1; i += 256)
    if (sh1[i]) atomicAdd(&hist1[(int64_t)h * kTokBins1 + i], sh1[i]);
}

// grid (H), 1024 threads.  idx[h][0..K): the K tokens with the largest keys, ascending; ties at the cut by lower index.
// Radix select in three digits (11 + 11 + 10 bits).  The histogram of the first digit over ALL keys comes from the probe pass
// (hist1: the probe kernel counts every key once with a shared-memory atomic), so the two histogram passes here only issue a
// shared-memory atomic for the keys that match the prefix found so far (a small fraction of N).  Every pass keeps eight independent loads in flight per thread (the keys are L2-resident; one
// CTA per head is latency-bound otherwise).  Histogram passes read strided (order does not matter), the compaction pass reads
// eight CONSECUTIVE keys per thread so that a block-wide scan of per-thread counts gives ordered output positions.
__global__ void __launch_bounds__(1024) token_topk_kernel(const uint32_t *__restrict__ keys, const uint32_t *__restrict__ hist1,
                                                          int32_t *__restrict__ idx, int64_t N, int K) {
  const int h = blockIdx.x;
  const uint32_t *key = keys + (int64_t)h * N;
  int32_t *out = idx + (int64_t)h * K;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __shared__ uint32_t hist[kTokBins1];
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t s_prefix, s_need;
  __shared__ int wtake[32], weq[32];
  uint32_t prefix = 0, mask = 0;
  int need = K;
  // digit d of `bits` bits at `shift`: hist[] holds the counts of the keys that match (prefix, mask); pick the bin, from the top,
  // in which the running count reaches `need` (block-wide: each thread owns two adjacent bins, suffix sums by warp scans)
  auto pick_bin = [&](int shift, int bins) {
    const int b0 = bins - 1 - 2 * (int)threadIdx.x, b1 = b0 - 1;  // descending bin order
    const uint32_t c0 = b0 >= 0 ? hist[b0] : 0u, c1 = b1 >= 0 ? hist[b1] : 0u;
    uint32_t inc = c0 + c1;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, off);
      if (lane >= off) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    uint32_t before = inc - (c0 + c1);  // keys in higher bins
    for (int w = 0; w < warp; ++w) before += wsum[w];
    if (before < (uint32_t)need && before + c0 + c1 >= (uint32_t)need) {  // exactly one thread
      const bool first = before + c0 >= (uint32_t)need;
      s_prefix = prefix | ((uint32_t)(first ? b0 : b1) << shift);
      s_need = (uint32_t)need - before - (first ? 0u : c0);
    }
    __syncthreads();
    prefix = s_prefix;
    need = (int)s_need;
    mask |= (uint32_t)(bins - 1) << shift;
    __syncthreads();
  };
  auto count_digit = [&](int shift, int bins) {
    for (int i = threadIdx.x; i < bins; i += 1024) hist[i] = 0u;
    __syncthreads();
    for (int64_t j0 = 0; j0 < N; j0 += 8 * 1024) {
      uint32_t kv[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int64_t j = j0 + threadIdx.x + 1024 * i;
        kv[i] = j < N ? __ldg(key + j) : 0u;
      }
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int64_t j = j0 + threadIdx.x + 1024 * i;
        if (j < N && (kv[i] & mask) == prefix) atomicAdd(&hist[(kv[i] >> shift) & (uint32_t)(bins - 1)], 1u);
      }
    }
    __syncthreads();
  };
  for (int i = threadIdx.x; i < kTokBins1; i += 1024) hist[i] = hist1[(int64_t)h * kTokBins1 + i];
  __syncthreads();
  pick_bin(21, 2048);
  count_digit(10, 2048);
  pick_bin(10, 2048);
  count_digit(0, 1024);
  pick_bin(0, 1024);
  const uint32_t tau = prefix;  // K-th largest key; take all keys above it and the first `need` (by index) equal to it
  int written = 0, eq_seen = 0;
  for (int64_t j0 = 0; j0 < N; j0 += 8 * 1024) {
    const int64_t jb = j0 + 8 * (int64_t)threadIdx.x;  // this thread's eight consecutive keys
    uint32_t kv[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) kv[i] = jb + i < N ? __ldg(key + jb + i) : 0u;
    int n_eq = 0, n_gt = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool in = jb + i < N;
      n_eq += (in && kv[i] == tau) ? 1 : 0;
      n_gt += (in && kv[i] > tau) ? 1 : 0;
    }
    // block-wide exclusive scan of the tie counts (needed to decide which ties are among the first `need`)
    int eq_inc = n_eq;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, eq_inc, off);
      if (lane >= off) eq_inc += t;
    }
    if (lane == 31) weq[warp] = eq_inc;
    __syncthreads();
    int eq_before = eq_seen + eq_inc - n_eq, eq_total = 0;
    for (int w = 0; w < 32; ++w) {
      if (w < warp) eq_before += weq[w];
      eq_total += weq[w];
    }
    int n_take = n_gt, eq_room = need - eq_before;  // ties this thread may still take
    if (eq_room < 0) eq_room = 0;
    n_take += n_eq < eq_room ? n_eq : eq_room;
    int tk_inc = n_take;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, tk_inc, off);
      if (lane >= off) tk_inc += t;
    }
    if (lane == 31) wtake[warp] = tk_inc;
    __syncthreads();
    int pos = written + tk_inc - n_take, total = 0;
    for (int w = 0; w < 32; ++w) {
      if (w < warp) pos += wtake[w];
      total += wtake[w];
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool in = jb + i < N;
      bool take = in && kv[i] > tau;
      if (in && kv[i] == tau) {
        if (eq_room > 0) { take = true; --eq_room; }
      }
      if (take) out[pos++] = (int32_t)(jb + i);
    }
    written += total;
    eq_seen += eq_total;
    __syncthreads();
  }
}

// grid (ceil(K / 32), H, 2): rows idx[h][i] of K (z = 0) / V (z = 1) -> compact [H][K][64] bf16.
__global__ void __launch_bounds__(256) token_gather_kernel(const __nv_bfloat16 *__restrict__ k, const __nv_bfloat16 *__restrict__ v,
                                                           const int32_t *__restrict__ idx, __nv_bfloat16 *__restrict__ kc,
                                                           __nv_bfloat16 *__restrict__ vc, SelGeom g, int K) {
  const int h = blockIdx.y;
  const int sub = threadIdx.x & 7, row = threadIdx.x >> 3;
  const int i = blockIdx.x * 32 + row;
  if (i >= K) return;
  const int64_t t = idx[(int64_t)h * K + i];
  const __nv_bfloat16 *src = (blockIdx.z ? v : k) + (int64_t)h * g.stride_head + t * g.stride_token + sub * 8;
  __nv_bfloat16 *dst = (blockIdx.z ? vc : kc) + ((int64_t)h * K + i) * 64 + sub * 8;
  *reinterpret_cast<uint4 *>(dst) = *reinterpret_cast<const uint4 *>(src);
}

// ------------------------------------------------------------------------------------------------ static broadcast (NEXT-4)
// Static kernel, second pattern of PAPER.md:L96 ("broadcasting the first frame's local attention map to other frames for
// cross-view interaction"; DESIGN reading A18): every T x T image block of the N x N attention map equals frame 0's local map
// P0 = softmax(Q0 K0^T / sqrt(D)), so a query at (frame f, position p) gets o = sum_p' P0[p][p'] * vbar[p'] with
// vbar[p'] = (1/S) sum_g v[g][p'] - the same row for every frame.  O(T^2 D + N D) instead of O(N^2 D).
//   frame_mean_kernel       vbar (bf16, RNE) and a compact copy of K0: grid (ceil(T/32), H, 2), 8 lanes per token row
//   (dense mode of saf3r_attn_kernel over (Q0, K0, vbar) writes frame 0's rows of out)
//   frame_broadcast_kernel  frame 0's rows of out (and lse) -> frames 1..S-1
__global__ void __launch_bounds__(256) frame_mean_kernel(const __nv_bfloat16 *__restrict__ k, const __nv_bfloat16 *__restrict__ v,
                                                         __nv_bfloat16 *__restrict__ kc, __nv_bfloat16 *__restrict__ vc, SelGeom g) {
  const int h = blockIdx.y, sub = threadIdx.x & 7, row = threadIdx.x >> 3;
  const int p = blockIdx.x * 32 + row;
  if (p >= g.T) return;
  __nv_bfloat16 *dst = (blockIdx.z ? vc : kc) + ((int64_t)h * g.T + p) * 64 + sub * 8;
  if (blockIdx.z == 0) {
    *reinterpret_cast<uint4 *>(dst) = *reinterpret_cast<const uint4 *>(k + (int64_t)h * g.stride_head + (int64_t)p * g.stride_token + sub * 8);
    return;
  }
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  const __nv_bfloat16 *src = v + (int64_t)h * g.stride_head + (int64_t)p * g.stride_token + sub * 8;
  for (int f0 = 0; f0 < g.S; f0 += 8) {  // frames in order, eight loads in flight
    uint4 raw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      raw[i] = make_uint4(0, 0, 0, 0);
      if (f0 + i < g.S) raw[i] = ld_stream_16(src + (int64_t)(f0 + i) * g.T * g.stride_token);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      float x[8];
      bf16x8_to_f32(raw[i], x);
#pragma unroll
      for (int c = 0; c < 8; ++c) acc[c] += x[c];
    }
  }
  const float inv = 1.f / (float)g.S;
  uint4 o;
  o.x = pack_bf16x2(acc[0] * inv, acc[1] * inv);
  o.y = pack_bf16x2(acc[2] * inv, acc[3] * inv);
  o.z = pack_bf16x2(acc[4] * inv, acc[5] * inv);
  o.w = pack_bf16x2(acc[6] * inv, acc[7] * inv);
  *reinterpret_cast<uint4 *>(dst) = o;
}

// grid (ceil(T / rows), S, H), rows = 256 / (16-byte chunks per output row: 8 for bf16, 16 for fp32).  Frames f >= 1 copy frame
// 0's output row; every frame's lse = lse0 + ln S (the partition function of the full row is S times frame 0's).
__global__ void __launch_bounds__(256) frame_broadcast_kernel(uint8_t *__restrict__ out, float *__restrict__ lse, const float *__restrict__ lse0,
                                                              SelGeom g, int64_t out_stride_head, int64_t out_stride_token, int elem_bytes) {
  const int h = blockIdx.z, f = blockIdx.y;
  const int chunks = 4 * elem_bytes;
  const int rows_per_cta = 256 / chunks;
  const int p = blockIdx.x * rows_per_cta + threadIdx.x / chunks, c = threadIdx.x % chunks;
  if (p >= g.T) return;
  if (f >= 1) {
    const uint8_t *src = out + ((int64_t)h * out_stride_head + (int64_t)p * out_stride_token) * elem_bytes + c * 16;
    uint8_t *dst = out + ((int64_t)h * out_stride_head + ((int64_t)f * g.T + p) * out_stride_token) * elem_bytes + c * 16;
    *reinterpret_cast<uint4 *>(dst) = *reinterpret_cast<const uint4 *>(src);
  }
  if (lse != nullptr && c == 0) lse[(int64_t)h * g.N + (int64_t)f * g.T + p] = lse0[(int64_t)h * g.T + p] + logf((float)g.S);
}

// ------------------------------------------------------------------------------------------------ Eq. 1 (NEXT-3)
// num[h] += sum (o_full - o_sparse)^2, den[h] += sum o_full^2 over one head's [N][64] outputs (bf16 or fp32), double accumulators;
// E(c) = num / den (Eq. 1).  grid (chunks, H), 256 threads, grid-stride over 16-byte chunks, one atomicAdd(double)
// pair per CTA (the two sums are order-dependent only in the last bits of a double).
__global__ void __launch_bounds__(256) nmse_kernel(const uint8_t *__restrict__ a, const uint8_t *__restrict__ b, int64_t N, int64_t stride_head,
                                                   int64_t stride_token, int is_fp32, double *__restrict__ num, double *__restrict__ den) {
  const int h = blockIdx.y;
  const int per_row = is_fp32 ? 16 : 8;  // 16-byte chunks per 64-element row
  const int esz = is_fp32 ? 4 : 2;
  double n = 0.0, d = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < N * per_row; i += (int64_t)gridDim.x * 256) {
    const int64_t off = ((int64_t)h * stride_head + (i / per_row) * stride_token) * esz + (i % per_row) * 16;
    const uint4 ra = *reinterpret_cast<const uint4 *>(a + off), rb = *reinterpret_cast<const uint4 *>(b + off);
    if (is_fp32) {
      const float fa[4] = {__uint_as_float(ra.x), __uint_as_float(ra.y), __uint_as_float(ra.z), __uint_as_float(ra.w)};
      const float fb[4] = {__uint_as_float(rb.x), __uint_as_float(rb.y), __uint_as_float(rb.z), __uint_as_float(rb.w)};
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const double x = fa[c], y = fb[c];
        n += (x - y) * (x - y);
        d += x * x;
      }
    } else {
      float fa[8], fb[8];
      bf16x8_to_f32(ra, fa);
      bf16x8_to_f32(rb, fb);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const double x = fa[c], y = fb[c];
        n += (x - y) * (x - y);
        d += x * x;
      }
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    n += __shfl_xor_sync(0xffffffffu, n, off);
    d += __shfl_xor_sync(0xffffffffu, d, off);
  }
  __shared__ double sn[8], sd[8];
  if ((threadIdx.x & 31) == 0) { sn[threadIdx.x >> 5] = n; sd[threadIdx.x >> 5] = d; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tn = 0.0, td = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { tn += sn[w]; td += sd[w]; }
    atomicAdd(num + h, tn);
    atomicAdd(den + h, td);
  }
}

}  // namespace saf3r
