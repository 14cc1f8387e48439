// Block-sparse / dense softmax attention for sm_100a (step a-4 / a-5 of DESIGN.md).
//
// One CTA per (head h, q-block I), two CTAs resident per SM (one CTA's softmax overlaps the other's MMAs).  Warps:
//   warps 0-3  softmax: thread r owns q-row r (= TMEM lane r).  One pass: S (fp32, TMEM) -> registers, row max
//              (lazy: the running max only moves when it grows by more than 2^8), p = exp2(s*c - m*c), row sum,
//              P (bf16) -> TMEM.  O is rescaled in TMEM only when the max moved.
//   warp  4    TMA producer: Q tile once, then one (K_J, V_J) tile pair per list entry into a 3-stage ring
//   warp  5    TMEM allocator + MMA issuer (one thread): S = Q K_J^T (tcgen05 SS), O += P V_J (tcgen05 TS: P from TMEM)
// TMEM columns: S [0,B) fp32, O [128,192) fp32, P [192,192+B/2) packed bf16.
#pragma once
#include "ptx.cuh"
#include "saf3r.h"

namespace saf3r {

struct AttnParams {
  const int64_t *row_ptr;  // [H*NB+1] or nullptr in dense mode
  const int32_t *col_idx;
  void *out;
  float *lse;  // [H][N] or nullptr
  int64_t out_stride_head, out_stride_token;
  int32_t N, NB, H;
  int32_t out_fp32;
  float scale_log2;  // (1/sqrt(D)) * log2(e)
  uint8_t head_order[SAF3R_MAX_HEADS];  // blockIdx.y -> head, longest lists first
};

constexpr int kD = 64;  // head_dim (bf16: one 128-byte swizzle row)
constexpr int kAttnThreads = 192;
constexpr int kStages = 3;
constexpr int kTmemCols = 256;
constexpr int kTmemO = 128;  // first O column
constexpr int kTmemP = 192;  // first P column
constexpr float kLazyLog2 = 8.f;  // rescale only when the row max grows by more than 2^8 (in exp2 units)

template <int B>
struct AttnSmem {
  static constexpr int kQ = 0;                       // 128 x 64 bf16 (only the first B rows are loaded)
  static constexpr int kK = kQ + 128 * 128;          // kStages x (B x 64 bf16)
  static constexpr int kV = kK + kStages * B * 128;
  static constexpr int kBar = kV + kStages * B * 128;
  static constexpr int kTotal = kBar + 128;
};

template <int B>
__global__ void __launch_bounds__(kAttnThreads, 2)
saf3r_attn_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                  const __grid_constant__ CUtensorMap map_v, const AttnParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  using L = AttnSmem<B>;
  const uint32_t sbase = smem_u32(smem);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int I = blockIdx.x, h = p.head_order[blockIdx.y];

  const uint32_t bar = sbase + L::kBar;
  const uint32_t bar_q = bar + 0;
  const uint32_t bar_kv_full = bar + 8;    // [kStages]
  const uint32_t bar_kv_empty = bar + 32;  // [kStages]
  const uint32_t bar_s_full = bar + 56;    // MMA -> softmax: S(e) is in TMEM
  const uint32_t bar_s_free = bar + 64;    // softmax -> MMA: S(e) has been read into registers (128 arrivals)
  const uint32_t bar_p_full = bar + 72;    // softmax -> MMA: P(e) is in TMEM, O rescaled (128 arrivals)
  const uint32_t bar_o_done = bar + 80;    // MMA -> softmax: PV(e) complete
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::kBar + 96);

  int64_t e0 = 0;
  int n_ent = p.NB;
  if (p.row_ptr != nullptr) {
    const int64_t r = (int64_t)h * p.NB + I;
    e0 = p.row_ptr[r];
    n_ent = (int)(p.row_ptr[r + 1] - e0);
  }

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();  // SWIZZLE_128B tiles need a 1024-byte aligned base
    mbar_init(bar_q, 1);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_kv_full + 8 * s, 1);
      mbar_init(bar_kv_empty + 8 * s, 1);
    }
    mbar_init(bar_s_full, 1);
    mbar_init(bar_s_free, 128);
    mbar_init(bar_p_full, 128);
    mbar_init(bar_o_done, 1);
    fence_mbar_init();
  }
  if (warp == 5) {
    tmem_alloc(smem_u32(tmem_slot), kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == 4) {
    // ------------------------------------------------------------ TMA producer
    if (lane == 0 && n_ent > 0) {
      tma_prefetch_desc(&map_q);
      tma_prefetch_desc(&map_k);
      tma_prefetch_desc(&map_v);
      mbar_arrive_expect_tx(bar_q, B * 128);
      tma_load_3d(sbase + L::kQ, &map_q, bar_q, 0, I * B, h);
      int Jn = p.row_ptr ? p.col_idx[e0] : 0;
      int s = 0, ph = 0;
      for (int e = 0; e < n_ent; ++e) {
        const int J = Jn;
        if (e + 1 < n_ent) Jn = p.row_ptr ? p.col_idx[e0 + e + 1] : e + 1;
        mbar_wait(bar_kv_empty + 8 * s, ph ^ 1);
        mbar_arrive_expect_tx(bar_kv_full + 8 * s, 2 * B * 128);
        tma_load_3d(sbase + L::kK + s * B * 128, &map_k, bar_kv_full + 8 * s, 0, J * B, h);
        tma_load_3d(sbase + L::kV + s * B * 128, &map_v, bar_kv_full + 8 * s, 0, J * B, h);
        if (++s == kStages) { s = 0; ph ^= 1; }
      }
    }
  } else if (warp == 5) {
    // ------------------------------------------------------------ MMA issuer
    if (lane == 0 && n_ent > 0) {
      constexpr uint32_t idesc_qk = umma_idesc_bf16(B, false);
      constexpr uint32_t idesc_pv = umma_idesc_bf16(kD, true);
      const uint64_t qdesc = umma_desc_sw128(sbase + L::kQ);
      const uint32_t tS = tmem, tO = tmem + kTmemO, tP = tmem + kTmemP;
      int sq = 0, phq = 0;  // stage / phase of the next QK
      auto issue_qk = [&]() {
        mbar_wait(bar_kv_full + 8 * sq, phq);
        tc_fence_after();
        const uint64_t kdesc = umma_desc_sw128(sbase + L::kK + sq * B * 128);
#pragma unroll
        for (int k = 0; k < kD / 16; ++k) umma_ss(tS, qdesc + 2 * k, kdesc + 2 * k, idesc_qk, k > 0);
        umma_commit(bar_s_full);
        if (++sq == kStages) { sq = 0; phq ^= 1; }
      };
      mbar_wait(bar_q, 0);
      issue_qk();
      int sv = 0;
      for (int e = 0; e < n_ent; ++e) {
        if (e + 1 < n_ent) {
          mbar_wait(bar_s_free, e & 1);  // S(e) is in registers -> overwrite it with S(e+1) while softmax(e) runs
          issue_qk();
        }
        mbar_wait(bar_p_full, e & 1);
        tc_fence_after();
        const uint64_t vdesc = umma_desc_sw128(sbase + L::kV + sv * B * 128);
#pragma unroll
        for (int kk = 0; kk < B / 16; ++kk)
          umma_ts(tO, tP + kk * 8, vdesc + (uint64_t)kk * 128, idesc_pv, (e > 0 || kk > 0) ? 1u : 0u);
        umma_commit(bar_kv_empty + 8 * sv);
        umma_commit(bar_o_done);
        if (++sv == kStages) sv = 0;
      }
    }
  } else {
    // ------------------------------------------------------------ softmax warps (thread r <-> q-row r)
    const int r = threadIdx.x;
    const uint32_t lane_off = (uint32_t)(warp * 32) << 16;
    const uint32_t tS = tmem + lane_off, tO = tmem + lane_off + kTmemO, tP = tmem + lane_off + kTmemP;
    const int tail = p.N - (p.NB - 1) * B;  // valid keys in the last k-block
    const int64_t tok = (int64_t)I * B + r;
    const bool row_valid = (r < B) && (tok < p.N);
    const float c = p.scale_log2;
    const float lazy_raw = kLazyLog2 / c;  // threshold on the raw logits
    float m = -INFINITY, l = 0.f;
    const int J_last = (n_ent > 0) ? (p.row_ptr ? p.col_idx[e0 + n_ent - 1] : p.NB - 1) : -1;
    const bool last_is_tail = (J_last == p.NB - 1) && (tail < B);

    for (int e = 0; e < n_ent; ++e) {
      uint32_t v[B];
      mbar_wait(bar_s_full, e & 1);
      tc_fence_after();
#pragma unroll
      for (int cb = 0; cb < B; cb += 32) tmem_ld32(tS + cb, *reinterpret_cast<uint32_t(*)[32]>(&v[cb]));
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(bar_s_free);
      if (e == n_ent - 1 && last_is_tail) {
#pragma unroll
        for (int i = 0; i < B; ++i)
          if (i >= tail) v[i] = 0xff800000u;  // -inf
      }
      // row max (3-input max)
      float mx0 = __uint_as_float(v[0]), mx1 = __uint_as_float(v[1]);
#pragma unroll
      for (int i = 2; i < B; i += 4) {
        mx0 = max3(mx0, __uint_as_float(v[i]), __uint_as_float(v[i + 1]));
        if (i + 3 < B) mx1 = max3(mx1, __uint_as_float(v[i + 2]), __uint_as_float(v[i + 3]));
      }
      const float mx = fmaxf(mx0, mx1);
      // lazy running max: move it only when some row of the warp grew by more than 2^8
      float alpha = 1.f;
      const bool moved = __any_sync(0xffffffffu, mx > m + lazy_raw);
      if (moved) {
        const float m_new = fmaxf(m, mx);
        alpha = ex2_approx((m - m_new) * c);
        m = m_new;
      }
      const float nmc = -m * c;
      // p = exp2(s*c - m*c); row sum; pack to bf16
      uint32_t pk[B / 2];
      uint64_t acc0 = 0ull, acc1 = 0ull;  // two packed fp32x2 partial sums
      const uint64_t c2 = pack_f32x2(c, c), nmc2 = pack_f32x2(nmc, nmc);
#pragma unroll
      for (int i = 0; i < B; i += 4) {
        float x0, x1, x2, x3;
        unpack_f32x2(fma_f32x2(pack_f32x2(__uint_as_float(v[i]), __uint_as_float(v[i + 1])), c2, nmc2), x0, x1);
        unpack_f32x2(fma_f32x2(pack_f32x2(__uint_as_float(v[i + 2]), __uint_as_float(v[i + 3])), c2, nmc2), x2, x3);
        x0 = ex2_approx(x0); x1 = ex2_approx(x1); x2 = ex2_approx(x2); x3 = ex2_approx(x3);
        acc0 = add_f32x2(acc0, pack_f32x2(x0, x1));
        acc1 = add_f32x2(acc1, pack_f32x2(x2, x3));
        pk[i >> 1] = pack_bf16x2(x0, x1);
        pk[(i >> 1) + 1] = pack_bf16x2(x2, x3);
      }
      float s0, s1, s2, s3;
      unpack_f32x2(acc0, s0, s1);
      unpack_f32x2(acc1, s2, s3);
      l = l * alpha + ((s0 + s1) + (s2 + s3));
      // PV(e-1) must be complete before P is overwritten and O is rescaled
      if (e > 0) {
        mbar_wait(bar_o_done, (e - 1) & 1);
        tc_fence_after();
        if (moved) {
#pragma unroll
          for (int cb = 0; cb < kD; cb += 32) {
            uint32_t o[32];
            tmem_ld32(tO + cb, o);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st32(tO + cb, o);
          }
        }
      }
#pragma unroll
      for (int cb = 0; cb < B / 2; cb += 32) tmem_st32(tP + cb, *reinterpret_cast<uint32_t(*)[32]>(&pk[cb]));
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(bar_p_full);
    }

    // ------------------------------------------------------------ epilogue: O / l -> global
    if (n_ent > 0) {
      mbar_wait(bar_o_done, (n_ent - 1) & 1);
      tc_fence_after();
    }
    const float inv_l = (n_ent > 0) ? 1.f / l : 0.f;
    uint8_t *orow = reinterpret_cast<uint8_t *>(p.out) +
                    ((int64_t)h * p.out_stride_head + tok * p.out_stride_token) * (p.out_fp32 ? 4 : 2);
#pragma unroll 1
    for (int cb = 0; cb < kD; cb += 32) {
      uint32_t v[32];
      if (n_ent > 0) {
        tmem_ld32(tO + cb, v);
        tmem_ld_wait();
      } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] = 0u;
      }
      if (row_valid) {
        if (p.out_fp32) {
          float4 *dst = reinterpret_cast<float4 *>(orow + cb * 4);
#pragma unroll
          for (int i = 0; i < 32; i += 4)
            dst[i >> 2] = make_float4(__uint_as_float(v[i]) * inv_l, __uint_as_float(v[i + 1]) * inv_l,
                                      __uint_as_float(v[i + 2]) * inv_l, __uint_as_float(v[i + 3]) * inv_l);
        } else {
          uint4 *dst = reinterpret_cast<uint4 *>(orow + cb * 2);
#pragma unroll
          for (int i = 0; i < 32; i += 8)
            dst[i >> 3] = make_uint4(pack_bf16x2(__uint_as_float(v[i]) * inv_l, __uint_as_float(v[i + 1]) * inv_l),
                                     pack_bf16x2(__uint_as_float(v[i + 2]) * inv_l, __uint_as_float(v[i + 3]) * inv_l),
                                     pack_bf16x2(__uint_as_float(v[i + 4]) * inv_l, __uint_as_float(v[i + 5]) * inv_l),
                                     pack_bf16x2(__uint_as_float(v[i + 6]) * inv_l, __uint_as_float(v[i + 7]) * inv_l));
        }
      }
    }
    if (row_valid && p.lse != nullptr)
      p.lse[(int64_t)h * p.N + tok] = (n_ent > 0) ? (m * c + log2f(l)) * 0.69314718055994531f : -INFINITY;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 5) {
    __syncwarp();
    tmem_dealloc(tmem, kTmemCols);
  }
}

}  // namespace saf3r
