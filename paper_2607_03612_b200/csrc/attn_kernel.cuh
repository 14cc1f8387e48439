// Block-sparse / dense softmax attention for sm_100a (step a-4 / a-5 of DESIGN.md).
//
// One CTA per (head h, q-block I).  Six warps:
//   warps 0-3  softmax: thread r owns q-row r (= TMEM lane r): reads S from TMEM, online softmax, writes P (bf16) to smem
//   warp  4    TMA producer: Q tile once, then one (K_J, V_J) tile pair per list entry into a 2-stage ring
//   warp  5    TMEM allocator + MMA issuer (one thread): S = Q K_J^T (tcgen05, SS) ; O += P V_J (tcgen05, SS)
// Accumulators live in TMEM: S at columns [0,B), O at columns [128,192).  Two CTAs are resident per SM, so one CTA's
// softmax overlaps the other's MMAs.
#pragma once
#include "ptx.cuh"

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
};

constexpr int kD = 64;            // head_dim (bf16: one 128-byte swizzle row)
constexpr int kAttnThreads = 192;
constexpr int kStages = 2;
constexpr int kTmemCols = 256;
constexpr int kTmemO = 128;       // first O column

template <int B>
struct AttnSmem {
  static constexpr int kQ = 0;                               // 128 x 64 bf16 (only the first B rows are loaded)
  static constexpr int kK = kQ + 128 * 128;                  // kStages x (B x 64 bf16)
  static constexpr int kV = kK + kStages * B * 128;
  static constexpr int kP = kV + kStages * B * 128;          // B/64 atoms of [128 rows][64 keys] bf16
  static constexpr int kBar = kP + 128 * B * 2;
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
  const int I = blockIdx.x, h = blockIdx.y;

  // barriers
  const uint32_t bar = sbase + L::kBar;
  const uint32_t bar_q = bar + 0;
  const uint32_t bar_kv_full = bar + 8;    // [kStages]
  const uint32_t bar_kv_empty = bar + 24;  // [kStages]
  const uint32_t bar_s_full = bar + 40;
  const uint32_t bar_p_full = bar + 48;
  const uint32_t bar_o_done = bar + 56;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::kBar + 64);

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
      for (int e = 0; e < n_ent; ++e) {
        const int s = e % kStages, n = e / kStages;
        const int J = Jn;
        if (e + 1 < n_ent) Jn = p.row_ptr ? p.col_idx[e0 + e + 1] : e + 1;
        mbar_wait(bar_kv_empty + 8 * s, (n & 1) ^ 1);
        mbar_arrive_expect_tx(bar_kv_full + 8 * s, 2 * B * 128);
        tma_load_3d(sbase + L::kK + s * B * 128, &map_k, bar_kv_full + 8 * s, 0, J * B, h);
        tma_load_3d(sbase + L::kV + s * B * 128, &map_v, bar_kv_full + 8 * s, 0, J * B, h);
      }
    }
  } else if (warp == 5) {
    // ------------------------------------------------------------ MMA issuer
    if (lane == 0 && n_ent > 0) {
      constexpr uint32_t idesc_qk = umma_idesc_bf16(B, false);
      constexpr uint32_t idesc_pv = umma_idesc_bf16(kD, true);
      const uint64_t qdesc = umma_desc_sw128(sbase + L::kQ);
      const uint32_t tS = tmem, tO = tmem + kTmemO;
      auto issue_qk = [&](int e) {
        const int s = e % kStages, n = e / kStages;
        mbar_wait(bar_kv_full + 8 * s, n & 1);
        tc_fence_after();
        const uint64_t kdesc = umma_desc_sw128(sbase + L::kK + s * B * 128);
#pragma unroll
        for (int k = 0; k < kD / 16; ++k) umma_ss(tS, qdesc + 2 * k, kdesc + 2 * k, idesc_qk, k > 0);
        umma_commit(bar_s_full);
      };
      mbar_wait(bar_q, 0);
      issue_qk(0);
      for (int e = 0; e < n_ent; ++e) {
        const int s = e % kStages;
        // P(e) is in smem and S has been read  ->  S may be overwritten by QK(e+1), then O += P(e) V(e)
        mbar_wait(bar_p_full, e & 1);
        tc_fence_after();
        if (e + 1 < n_ent) issue_qk(e + 1);
        const uint64_t vdesc = umma_desc_sw128(sbase + L::kV + s * B * 128);
#pragma unroll
        for (int kk = 0; kk < B / 16; ++kk) {
          const uint64_t pdesc = umma_desc_sw128(sbase + L::kP + (kk / 4) * (128 * 128) + (kk % 4) * 32);
          umma_ss(tO, pdesc, vdesc + (uint64_t)kk * 128, idesc_pv, (e > 0 || kk > 0) ? 1u : 0u);
        }
        umma_commit(bar_kv_empty + 8 * s);
        umma_commit(bar_o_done);
      }
    }
  } else {
    // ------------------------------------------------------------ softmax warps (thread r <-> q-row r)
    const int r = threadIdx.x;
    const uint32_t lane_off = (uint32_t)(warp * 32) << 16;
    const uint32_t tS = tmem + lane_off, tO = tmem + lane_off + kTmemO;
    const int tail = p.N - (p.NB - 1) * B;  // valid keys in the last k-block
    const int64_t tok = (int64_t)I * B + r;
    const bool row_valid = (r < B) && (tok < p.N);
    float m = -INFINITY, l = 0.f;
    const float c = p.scale_log2;
    const int J_last = (n_ent > 0) ? (p.row_ptr ? p.col_idx[e0 + n_ent - 1] : p.NB - 1) : -1;

    for (int e = 0; e < n_ent; ++e) {
      const int ncols = (e == n_ent - 1 && J_last == p.NB - 1) ? tail : B;
      mbar_wait(bar_s_full, e & 1);
      tc_fence_after();
      // pass 1: row max of the raw logits
      float mx = -INFINITY;
#pragma unroll 1
      for (int cb = 0; cb < B; cb += 32) {
        uint32_t v[32];
        tmem_ld32(tS + cb, v);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 32; ++i)
          if (cb + i < ncols) mx = fmaxf(mx, __uint_as_float(v[i]));
      }
      const float m_new = fmaxf(m, mx);
      const float alpha = ex2_approx((m - m_new) * c);
      const float mc = m_new * c;
      // PV(e-1) must be complete before P smem is overwritten and O is rescaled
      if (e > 0) {
        mbar_wait(bar_o_done, (e - 1) & 1);
        tc_fence_after();
      }
      // pass 2: p = exp2(s*c - m*c), row sum, P -> smem (K-major, 128B swizzle)
      float sum = 0.f;
#pragma unroll 1
      for (int cb = 0; cb < B; cb += 32) {
        uint32_t v[32];
        tmem_ld32(tS + cb, v);
        tmem_ld_wait();
        uint32_t pk[16];
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          float p0 = (cb + i < ncols) ? ex2_approx(fmaf(__uint_as_float(v[i]), c, -mc)) : 0.f;
          float p1 = (cb + i + 1 < ncols) ? ex2_approx(fmaf(__uint_as_float(v[i + 1]), c, -mc)) : 0.f;
          sum += p0 + p1;
          pk[i >> 1] = pack_bf16x2(p0, p1);
        }
        // keys cb..cb+31 of row r: atom = cb/64, 16-byte chunks ((cb%64)/8 .. +3), chunk index XOR (r%8)
        const uint32_t rowbase = sbase + L::kP + (cb >> 6) * (128 * 128) + (r >> 3) * 1024 + (r & 7) * 128;
#pragma unroll
        for (int q4 = 0; q4 < 4; ++q4) {
          const uint32_t chunk = (uint32_t)(((cb & 63) >> 3) + q4) ^ (uint32_t)(r & 7);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(rowbase + chunk * 16), "r"(pk[4 * q4]),
                       "r"(pk[4 * q4 + 1]), "r"(pk[4 * q4 + 2]), "r"(pk[4 * q4 + 3])
                       : "memory");
        }
      }
      l = l * alpha + sum;
      m = m_new;
      // rescale O (warp-uniform decision; tcgen05.ld/st are .sync.aligned)
      if (e > 0 && __any_sync(0xffffffffu, alpha != 1.f)) {
#pragma unroll 1
        for (int cb = 0; cb < kD; cb += 32) {
          uint32_t v[32];
          tmem_ld32(tO + cb, v);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * alpha);
          tmem_st32(tO + cb, v);
        }
        tmem_st_wait();
      }
      fence_proxy_async_smem();
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
  if (warp == 5) tmem_dealloc(tmem, kTmemCols);
}

}  // namespace saf3r
