// Token-wise per-frame Top-K (SURVEY 8(f) NEXT-2 iii): "compute the global cosine similarity between all
// patches, storing the indices of the per-frame Top-K matched patches ... cached and reused by all subsequent DINO Top-K kernels".
//   feat_rnorm_kernel        rn[t] = 1 / |f_t| (0 for a zero feature), one streaming pass over the per-sequence features
//   token_sim_kernel         a strip of the N x N cosine matrix on the tensor cores: one CTA = one 128 x 128 tile F_I F_J^T
//                            (TMA -> SW128 smem -> tcgen05.mma SS, fp32 in TMEM), epilogue scales column j by rn[j] and stores
//                            order-preserving uint32 keys (the factor 1/|f_i| is constant along a row and cannot change a ranking)
//   token_frame_topk_kernel  one warp per (query, frame): the atomics-free bisection top-n of select_kernels.cuh over the T keys of
//                            the frame -> K ascending token indices (ties by lower index, the oracle's total order)
//   token_union_kernel       per q-tile of B queries: the union of its queries' keys (a T-bit map per frame in shared memory),
//                            packed over the frames into tiles of B gathered keys, and the per-(query, key) bit masks the
//                            attention kernel applies before the row max (so that its tcgen05 tiles stay dense)
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"
#include "select_kernels.cuh"
#include "token_kernels.cuh"

namespace saf3r {

// grid ceil(N / 32), 256 threads: 8 lanes per 128-byte feature row
__global__ void __launch_bounds__(256) feat_rnorm_kernel(const __nv_bfloat16 *__restrict__ f, int64_t N, int64_t stride_token,
                                                         float *__restrict__ rn) {
  const int sub = threadIdx.x & 7;
  const int64_t t = (int64_t)blockIdx.x * 32 + (threadIdx.x >> 3);
  float ss = 0.f;
  if (t < N) {
    float x[8];
    bf16x8_to_f32(ld_stream_16(f + t * stride_token + sub * 8), x);
#pragma unroll
    for (int c = 0; c < 8; ++c) ss = fmaf(x[c], x[c], ss);
  }
  ss += __shfl_xor_sync(0xffffffffu, ss, 1);
  ss += __shfl_xor_sync(0xffffffffu, ss, 2);
  ss += __shfl_xor_sync(0xffffffffu, ss, 4);
  if (t < N && sub == 0) {
    const float n = sqrtf(ss);
    rn[t] = n < 1e-20f ? 0.f : 1.f / n;
  }
}

// grid (ceil(N / 128) key tiles, q-tiles of the strip), 128 threads.  keys: [strip rows][ld] uint32, row = 128 * blockIdx.y + r.
constexpr int kSimSmem = 2 * 128 * 128 + 512 + 64 + 1024;  // A tile, B tile, rn of the key tile, barriers; + alignment slack
__global__ void __launch_bounds__(128) token_sim_kernel(const __grid_constant__ CUtensorMap map_f, const float *__restrict__ rn,
                                                        uint32_t *__restrict__ keys, int64_t N, int64_t ld, int q_tile0) {
  extern __shared__ uint8_t sim_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(sim_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t sA = smem_u32(smem), sB = sA + 128 * 128;
  float *s_rn = reinterpret_cast<float *>(smem + 2 * 128 * 128);
  const uint32_t bar_ld = sA + 2 * 128 * 128 + 512, bar_mma = bar_ld + 8;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + 2 * 128 * 128 + 512 + 16);
  const int warp = threadIdx.x >> 5;
  const int J = blockIdx.x, I = q_tile0 + blockIdx.y;
  if (threadIdx.x == 0) {
    mbar_init(bar_ld, 1);
    mbar_init(bar_mma, 1);
    fence_mbar_init();
  }
  if (warp == 0) {
    tmem_alloc(smem_u32(tmem_slot), 128);
    tmem_relinquish();
  }
  {
    const int64_t j = (int64_t)J * 128 + threadIdx.x;
    s_rn[threadIdx.x] = j < N ? rn[j] : 0.f;
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  if (warp == 0) {
    if (elect_one_sync()) {
      mbar_arrive_expect_tx(bar_ld, 2 * 128 * 128);
      tma_load_3d(sA, &map_f, bar_ld, 0, I * 128, 0);
      tma_load_3d(sB, &map_f, bar_ld, 0, J * 128, 0);
    }
    __syncwarp();
    mbar_wait(bar_ld, 0);
    tc_fence_after();
    if (elect_one_sync()) {
      constexpr uint32_t idesc = umma_idesc_bf16(128, false);
      const uint64_t adesc = umma_desc_sw128(sA), bdesc = umma_desc_sw128(sB);
#pragma unroll
      for (int k = 0; k < 4; ++k) umma_ss(tmem, adesc + 2 * k, bdesc + 2 * k, idesc, k > 0);
      umma_commit(bar_mma);
    }
    __syncwarp();
  }
  mbar_wait(bar_mma, 0);
  tc_fence_after();
  const int r = threadIdx.x;  // TMEM lane = query row of the tile
  const uint32_t trow = tmem + ((uint32_t)(warp * 32) << 16);
  uint32_t *dst = keys + ((int64_t)blockIdx.y * 128 + r) * ld + (int64_t)J * 128;
#pragma unroll 1
  for (int cb = 0; cb < 128; cb += 16) {
    uint32_t v[16];
    tmem_ld16(trow + cb, v);
    tmem_ld_wait();
    uint32_t o[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) o[i] = score_key(__uint_as_float(v[i]) * s_rn[cb + i]);
#pragma unroll
    for (int i = 0; i < 16; i += 4) *reinterpret_cast<uint4 *>(dst + cb + i) = make_uint4(o[i], o[i + 1], o[i + 2], o[i + 3]);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 128);
}

// grid ceil(strip rows * S / 8), 256 threads: warp -> (row of the strip, frame).  idx: [N][S][K] int32.
__global__ void __launch_bounds__(256) token_frame_topk_kernel(const uint32_t *__restrict__ keys, int64_t ld, int64_t row0, int rows, int64_t N,
                                                               int S, int T, int K, int32_t *__restrict__ idx) {
  const int64_t w = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (w >= (int64_t)rows * S) return;
  const int r = (int)(w / S), g = (int)(w % S);
  const int64_t i = row0 + r;
  if (i >= N) return;
  warp_topn_bisect(keys + (int64_t)r * ld + (int64_t)g * T, T, K, idx + (i * S + g) * K, g * T);
}

// Union + masks of the q-tile blockIdx.x.  kFill = false: tiles[I + 1] = number of B-key tiles of the q-tile (scanned into tile_ptr
// afterwards).  kFill = true: key_idx / mask of those tiles (mask must be zero on entry).  Dynamic smem: 2 * ceil(T/32) words.
template <bool kFill>
__global__ void __launch_bounds__(256) token_union_kernel(const int32_t *__restrict__ idx, int64_t N, int S, int T, int K, int B,
                                                          int64_t *__restrict__ tile_ptr, int32_t *__restrict__ key_idx,
                                                          uint32_t *__restrict__ mask, int64_t capacity_tiles) {
  extern __shared__ uint32_t un_sm[];
  const int W = (T + 31) / 32;
  uint32_t *bm = un_sm, *pre = un_sm + W;
  __shared__ int s_total;
  const int I = blockIdx.x;
  const int64_t tile0 = kFill ? tile_ptr[I] : 0;
  if (kFill && tile_ptr[I + 1] > capacity_tiles) return;  // does not fit: the caller sees tile_ptr[last] > capacity
  int base = 0;
  for (int g = 0; g < S; ++g) {
    for (int w = threadIdx.x; w < W; w += 256) bm[w] = 0u;
    __syncthreads();
    for (int e = threadIdx.x; e < B * K; e += 256) {
      const int r = e / K;
      const int64_t i = (int64_t)I * B + r;
      if (i < N) {
        const int j = idx[(i * S + g) * K + (e % K)] - g * T;
        atomicOr(&bm[j >> 5], 1u << (j & 31));
      }
    }
    __syncthreads();
    if (threadIdx.x < 32) {  // exclusive prefix of the word popcounts
      int run = 0;
      for (int w0 = 0; w0 < W; w0 += 32) {
        const int w = w0 + threadIdx.x;
        const int c = w < W ? __popc(bm[w]) : 0;
        int inc = c;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
          const int t = __shfl_up_sync(0xffffffffu, inc, off);
          if ((int)threadIdx.x >= off) inc += t;
        }
        if (w < W) pre[w] = (uint32_t)(run + inc - c);
        run += __shfl_sync(0xffffffffu, inc, 31);
      }
      if (threadIdx.x == 0) s_total = run;
    }
    __syncthreads();
    if (kFill) {
      for (int w = threadIdx.x; w < W; w += 256) {
        uint32_t bits = bm[w];
        int64_t pos = tile0 * B + base + pre[w];
        while (bits) {
          const int b = __ffs(bits) - 1;
          bits &= bits - 1;
          key_idx[pos++] = g * T + w * 32 + b;
        }
      }
      for (int e = threadIdx.x; e < B * K; e += 256) {
        const int r = e / K;
        const int64_t i = (int64_t)I * B + r;
        if (i < N) {
          const int j = idx[(i * S + g) * K + (e % K)] - g * T;
          const int slot = base + (int)pre[j >> 5] + __popc(bm[j >> 5] & ((1u << (j & 31)) - 1u));
          const int64_t t = tile0 + slot / B;
          const int c = slot % B;
          atomicOr(&mask[(t * B + r) * (B / 32) + (c >> 5)], 1u << (c & 31));
        }
      }
    }
    base += s_total;
    __syncthreads();
  }
  const int tiles = (base + B - 1) / B;
  if (!kFill) {
    if (threadIdx.x == 0) tile_ptr[I + 1] = tiles;
  } else {
    for (int s = base + threadIdx.x; s < tiles * B; s += 256) key_idx[tile0 * B + s] = -1;  // padding of the last tile
  }
}

}  // namespace saf3r
