// Block-sparse / dense softmax attention for sm_100a (step a-4 / a-5 of DESIGN.md).
//
// One CTA per (head h, q-block I), two CTAs resident per SM.  At D = 64 the exponentials, not the tensor pipe, bound
// this kernel (16 384 exp per 128x128 tile against 16 MUFU lanes/clk/SM = 1024 clk, versus 512 clk of MMA), so the
// softmax of a tile is split by COLUMNS over two warp groups that use different pipes:
//   warps 0-3   "MUFU" softmax: thread r owns q-row r (TMEM lane r), the first kSplitLo / kSplitHi columns of the tile's two
//               64-key halves: p = ex2.approx(s*c - m*c)
//   warps 4-7   "FMA"  softmax: same rows, the other columns of each half: 2^x by Cody-Waite + degree-3 polynomial on the FMA/ALU
//               pipes (no MUFU).  The two halves of a row exchange their partial row max through shared memory.
//   warp  8     TMA producer: Q tile once, then K_J into a 3-stage ring and V_J into a 2-stage ring
//   warp  9     TMEM allocator + MMA issuer (one thread): S = Q K_J^T (tcgen05 SS); per 64-key half of P: O += P V_J and the row
//               sums l += P 1 (tcgen05 TS: P from TMEM; N = 16 all-ones B tile), so the softmax warps add nothing per element
//   warps 10-11 idle (they only complete the third warpgroup so that setmaxnreg can hand its registers over); in the token-list
//               mode warp 8 gathers the K tiles and warp 10 the V tiles with cp.async instead of TMA
// Running max is lazy (moves only when a row max grows by more than 2^8), so O in TMEM is rescaled rarely.  And it is
// FROZEN as soon as it provably cannot matter: by Cauchy-Schwarz every logit of row i is at most |q_i| * max_j |k_j| / sqrt(D)
// (kmax[h] = max_j |k_j| comes from knorm_kernel, one streaming pass over K before the launch).  Once that bound is within
// 2^kFreezeLog2 of the row's reference max for all 32 rows of a warp, no later tile can overflow (p <= 2^64, far inside the
// bf16 / fp32 exponent range) and none can underflow relative to the true max, so the remaining tiles skip the row-max pass,
// the exchange between the two halves and the named barrier altogether - about an eighth of the softmax instructions.
// TMEM columns: S [0,B) fp32, O [128,192) fp32, l [192,208) fp32, P [208,240): one 64-key half of the tile (packed bf16; of the second
// half only the FMA group's keys [96,128)), PB [240,256): the MUFU group's keys [64,96) of the second half.
#pragma once
#include <type_traits>

#include "ptx.cuh"
#include "saf3r.h"

namespace saf3r {

struct AttnParams {
  const int64_t *row_ptr;  // [H*NB+1] or nullptr in dense mode
  const int32_t *col_idx;
  void *out;
  float *lse;  // [H][N] or nullptr
  int64_t out_stride_head, out_stride_token;
  int32_t N, NB, H;      // query tokens / q-blocks / heads
  int32_t N_kv, NB_kv;  // key/value tokens / k-blocks (== N, NB except in the token-granular variants)
  int32_t out_fp32;
  float scale_log2;  // (1/sqrt(D)) * log2(e)
  const float *kmax;  // [H] max_j |k_j|_2 over the head's key tokens (knorm_kernel), or nullptr: never freeze the max
  const uint8_t *head_order;  // dev, blockIdx.y -> head, longest lists first (knorm_kernel); nullptr: identity
  // token-list mode (kTok; SURVEY 8(f) NEXT-2 iii): the k-tiles of q-tile I are tiles [tile_ptr[I], tile_ptr[I+1]) of B gathered key
  // tokens each (key_idx, -1 = padding), shared by all heads; mask bit (row r, column c) of a tile says whether query r keeps key c
  const int64_t *tile_ptr;
  const int32_t *key_idx;
  const uint32_t *mask;  // [tile][B rows][B/32 words]
  int64_t capacity_tiles;  // tiles key_idx / mask hold: a q-tile whose range ends beyond it (a short-capacity _fill left it unwritten) is skipped
  const __nv_bfloat16 *k_base, *v_base;
  int64_t kv_stride_head, kv_stride_token;
};

constexpr int kD = 64;  // head_dim (bf16: one 128-byte swizzle row)
constexpr int kAttnThreads = 384;
constexpr int kKStages = 3, kVStages = 2;
constexpr int kTmemCols = 256;
constexpr int kTmemO = 128;  // first O column (64 fp32 columns)
constexpr int kTmemL = 192;  // row sums of P: 16 identical fp32 columns written by the ones-MMA (column 0 is read)
constexpr int kTmemP = 208;  // P of ONE 64-key half of the tile, packed bf16 (32 columns)
constexpr float kLazyLog2 = 8.f;
constexpr int kSleepTma = 128, kSleepMma = 48;  // ns between two mbarrier polls of the producer / issuer warps
constexpr float kFreezeLog2 = 64.f;  // freeze the reference max when no logit can exceed it by more than 2^64
constexpr int kTmemPB = 240; // second P buffer (16 columns): the MUFU group's keys [64, 96) of the tile, so that the group on the critical path never waits for the first half's MMAs
constexpr int kSplitLo128 = 40, kSplitHi128 = 32;
static_assert(kSplitHi128 == 32, "the MUFU group's second-half keys must be exactly the two K = 16 steps that read kTmemPB");  // columns of the first / second 64-key half whose exponentials use the MUFU (rest: FMA-pipe polynomial); multiples of 8
constexpr int kRegsMufu = 112, kRegsFma = 88, kRegsIdle = 40;  // 128*(112+88+40) = 30720 = 384 threads * 80 registers

template <int B>
struct AttnSmem {
  static constexpr int split_of(int hh) { return (B == 128) ? (hh == 0 ? kSplitLo128 : kSplitHi128) : 32; }  // MUFU columns of half hh
  static constexpr int kQ = 0;                          // 128 x 64 bf16 (only the first B rows are loaded)
  static constexpr int kK = kQ + 128 * 128;             // kKStages x (B x 64 bf16)
  static constexpr int kV = kK + kKStages * B * 128;    // kVStages x (B x 64 bf16)
  static constexpr int kOnes = kV + kVStages * B * 128; // 16 x 64 bf16 ones (K-major B operand of the row-sum MMA; 1024-byte aligned)
  static constexpr int kMax = kOnes + 2048;             // float [2 parity][2 half][128 rows]
  static constexpr int kBar = kMax + 2 * 2 * 128 * 4;
  static constexpr int kTotal = kBar + 256;
};

// one softmax group: rows = TMEM lanes of this warp; of every 64-key half of the B-wide tile it owns the columns
// [C0h, C0h + NCH): the MUFU group the first kSplitHalf, the FMA group the rest.  P goes to TMEM one 64-key half at a time (the
// 32-column P buffer is handed back by the PV MMAs of the previous half), and the row sum of the bf16-ROUNDED weights is an MMA of
// its own (P x ones, N = 16) into kTmemL: no per-element add in these warps, and the sum matches what the PV product multiplies.
template <int B, bool kFma, bool kTok>
__device__ __forceinline__ void softmax_half(const AttnParams &p, uint8_t *smem, uint32_t tmem, int n_ent, int64_t e0, int h,
                                             int I, uint32_t bar_q, uint32_t bar_s_full, uint32_t bar_s_free,
                                             uint32_t bar_p_full /* [NH] */, uint32_t bar_pv0_done, uint32_t bar_o_done) {
  using L = AttnSmem<B>;
  constexpr int NH = B / 64;                       // 64-key halves of a tile
  // this group's columns of half hh: [64 hh + c0(hh), 64 hh + c0(hh) + nch(hh)); v[] holds half 0's columns, then half 1's
  auto c0 = [](int hh) constexpr { return kFma ? L::split_of(hh) : 0; };
  auto nch = [](int hh) constexpr { return kFma ? 64 - L::split_of(hh) : L::split_of(hh); };
  constexpr int NCH0 = nch(0), NCH1 = (NH == 2) ? nch(1) : 0;
  constexpr int NC = NCH0 + NCH1;
  static_assert(NCH0 % 8 == 0 && NCH0 > 0 && NCH0 < 64 && NCH1 % 8 == 0 && (NH == 1 || (NCH1 > 0 && NCH1 < 64)), "column split must be a multiple of 8");
  auto col_of = [&](int i) constexpr { return i < NCH0 ? c0(0) + i : 64 + c0(1) + (i - NCH0); };
  constexpr int kHalf = kFma ? 1 : 0;
  const int r = threadIdx.x & 127;
  const int pair_bar = 1 + (r >> 5);  // named barrier shared by the two warps that own these 32 rows
  // TMEM lane block of this warp; the shuffle makes it warp-uniform by construction so that ptxas keeps the tcgen05.ld/st
  // addresses in uniform registers instead of re-deriving them (R2UR) every iteration
  const uint32_t lane_off = (uint32_t)(__shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0) & 3) << 21;
  const uint32_t tS = tmem + lane_off, tO = tmem + lane_off + kTmemO + 32 * kHalf, tP = tmem + lane_off + kTmemP;
  const uint32_t tL = tmem + lane_off + kTmemL;
  float *smax = reinterpret_cast<float *>(smem + L::kMax);
  const int tail = p.N_kv - (p.NB_kv - 1) * B;  // valid keys in the last k-block
  const int64_t tok = (int64_t)I * B + r;
  const bool row_valid = (r < B) && (tok < p.N);
  const float c = p.scale_log2;
  const float lazy_raw = kLazyLog2 / c;
  float m = -INFINITY;
  const int J_last = (n_ent > 0 && !kTok) ? (p.row_ptr ? p.col_idx[e0 + n_ent - 1] : p.NB_kv - 1) : -1;
  const bool last_is_tail = !kTok && (J_last == p.NB_kv - 1) && (tail < B);
  // Cauchy-Schwarz bound of this row's logits (in the units of m: raw scores), from the Q tile in shared memory.  Both groups
  // of a row read the same eight 16-byte chunks in the same (physical) order, so they get the same bits and take the same
  // freeze decision without talking to each other.
  float bound = INFINITY;
  bool frozen = false, noclamp = false;
  if (p.kmax != nullptr && n_ent > 1) {
    mbar_wait(bar_q, 0);
    const uint4 *qrow = reinterpret_cast<const uint4 *>(smem + L::kQ + r * 128);
    float ss = 0.f;
#pragma unroll
    for (int ch = 0; ch < 8; ++ch) {
      const uint4 w = qrow[ch];
      const uint32_t u[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float lo = __uint_as_float(u[i] << 16), hi = __uint_as_float(u[i] & 0xffff0000u);
        ss = fmaf(lo, lo, ss);
        ss = fmaf(hi, hi, ss);
      }
    }
    bound = sqrtf(ss) * p.kmax[h] * 1.001f;  // rounding of the two norms and of the tensor-core sums: far below 1e-3
  }
  const float freeze_raw = kFreezeLog2 / c;

  for (int e = 0; e < n_ent; ++e) {
    uint32_t v[NC];  // v[i] = score of column col_of(i)
    mbar_wait(bar_s_full, e & 1);
    tc_fence_after();
    tmem_ld_n<NCH0>(tS + c0(0), v);
    if constexpr (NH == 2) tmem_ld_n<(NCH1 > 0 ? NCH1 : 8)>(tS + 64 + c0(1), &v[NCH0]);
    tmem_ld_wait();
    tc_fence_before();
    mbar_arrive(bar_s_free);
    if (e == n_ent - 1 && last_is_tail) {
#pragma unroll
      for (int i = 0; i < NC; ++i)
        if (col_of(i) >= tail) v[i] = 0xff800000u;  // -inf
    }
    if (kTok) {  // per-(query, key) mask of this tile: keys the query did not select get -inf before the max
      uint32_t mw[B / 32];
      const uint32_t *mrow = p.mask + ((e0 + e) * B + (r < B ? r : 0)) * (B / 32);
#pragma unroll
      for (int w = 0; w < B / 32; ++w) mw[w] = r < B ? __ldg(mrow + w) : 0u;
#pragma unroll
      for (int i = 0; i < NC; ++i) {
        const int col = col_of(i);
        if (!((mw[col / 32] >> (col & 31)) & 1u)) v[i] = 0xff800000u;
      }
    }
    float alpha = 1.f;
    bool moved = false;
    if (!frozen) {
      // partial row max over this group's columns, then exchange with the other group
      float mx0 = __uint_as_float(v[0]), mx1 = __uint_as_float(v[1]), mx2 = __uint_as_float(v[2]), mx3 = __uint_as_float(v[3]);
#pragma unroll
      for (int i = 4; i < NC; i += 8) {
        mx0 = max3(mx0, __uint_as_float(v[i]), __uint_as_float(v[i + 1]));
        mx1 = max3(mx1, __uint_as_float(v[i + 2]), __uint_as_float(v[i + 3]));
        if (i + 4 < NC) {
          mx2 = max3(mx2, __uint_as_float(v[i + 4]), __uint_as_float(v[i + 5]));
          mx3 = max3(mx3, __uint_as_float(v[i + 6]), __uint_as_float(v[i + 7]));
        }
      }
      float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
      float *slot = smax + (e & 1) * 256;
      slot[kHalf * 128 + r] = mx;
      named_bar_sync(pair_bar, 64);
      mx = fmaxf(mx, slot[(1 - kHalf) * 128 + r]);
      // lazy running max (identical decision in both groups: same rows, same combined max)
      moved = __any_sync(0xffffffffu, mx > m + lazy_raw);
      if (moved) {
        const float m_new = fmaxf(m, mx);
        alpha = ex2_approx((m - m_new) * c);
        if (kTok && m_new == -INFINITY) alpha = 1.f;  // this row has seen no kept key yet (another row of the warp moved)
        m = m_new;
      }
      // no later logit of these 32 rows can exceed m by more than 2^kFreezeLog2: m stays where it is from now on
      frozen = __all_sync(0xffffffffu, bound <= m + freeze_raw);
      if (kFma && frozen) noclamp = __all_sync(0xffffffffu, (bound + fabsf(m)) * c < 120.f);
    }
    const float nmc = (kTok && m == -INFINITY) ? 0.f : -m * c;  // a row without a kept key so far: every x stays -inf, p = 0
    const uint64_t c2 = pack_f32x2(c, c), nmc2 = pack_f32x2(nmc, nmc);
    // the polynomial group needs its argument clamped at -126 unless every x of the tile is known to be above it: frozen max,
    // |logit| <= bound for all 32 rows (Cauchy-Schwarz again: x >= -(bound + m) c), no masked (-inf) column in the tile
    const bool fast = kFma && !kTok && noclamp && !(e == n_ent - 1 && last_is_tail);
    uint32_t pk[(NCH0 > NCH1 ? NCH0 : NCH1) / 2];
    auto exp_half = [&](auto clamp_tag, auto hh_tag) {
      constexpr bool kClamp = decltype(clamp_tag)::value;
      constexpr int hh = decltype(hh_tag)::value;
#pragma unroll
      for (int j = 0; j < nch(hh) / 2; ++j) {
        const uint64_t x2 =
            fma_f32x2(pack_f32x2(__uint_as_float(v[hh * NCH0 + 2 * j]), __uint_as_float(v[hh * NCH0 + 2 * j + 1])), c2, nmc2);
        float p0, p1;
        if (kFma) {
          exp2_emu_f32x2<kClamp>(x2, p0, p1);
        } else {
          unpack_f32x2(x2, p0, p1);
          p0 = ex2_approx(p0);
          p1 = ex2_approx(p1);
        }
        pk[j] = pack_bf16x2(p0, p1);
      }
    };
    auto do_half = [&](auto hh_tag) {
      constexpr int hh = decltype(hh_tag)::value;
      if (fast) exp_half(std::false_type{}, hh_tag);
      else exp_half(std::true_type{}, hh_tag);
      if (hh == 0) {
        // PV(e-1) must be complete before the P buffer is overwritten and O / the row sum are rescaled
        if (e > 0) {
          mbar_wait(bar_o_done, (e - 1) & 1);
          tc_fence_after();
          if (moved) {  // this group rescales its 32 of the 64 O columns (the MUFU group also the row sum)
            uint32_t o[32];
            uint32_t lsum = 0;
            tmem_ld32(tO, o);
            if (!kFma) tmem_ld1(tL, lsum);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st32(tO, o);
            if (!kFma) tmem_st1(tL, __float_as_uint(__uint_as_float(lsum) * alpha));
          }
        }
      } else {
        if (kFma || NH == 1) {
          mbar_wait(bar_pv0_done, e & 1);  // the MMAs of the first half have read the P buffer
          tc_fence_after();
        }
      }
      if (hh == 1 && !kFma) tmem_st_n<nch(hh) / 2>(tmem + lane_off + kTmemPB, pk);   // the MUFU group's second-half keys [64, 96): a buffer of their own
      else tmem_st_n<nch(hh) / 2>(tP + c0(hh) / 2, pk);
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(bar_p_full + 8 * hh);
    };
    do_half(std::integral_constant<int, 0>{});
    if constexpr (NH == 2) do_half(std::integral_constant<int, 1>{});
  }

  // ------------------------------------------------------------ epilogue: O / l -> global (32 of the 64 columns each)
  if (n_ent > 0) {
    mbar_wait(bar_o_done, (n_ent - 1) & 1);
    tc_fence_after();
  }
  uint8_t *orow = reinterpret_cast<uint8_t *>(p.out) +
                  ((int64_t)h * p.out_stride_head + tok * p.out_stride_token + 32 * kHalf) * (p.out_fp32 ? 4 : 2);
  uint32_t o[32];
  uint32_t lbits = 0;
  if (n_ent > 0) {
    tmem_ld32(tO, o);
    tmem_ld1(tL, lbits);
    tmem_ld_wait();
  } else {
#pragma unroll
    for (int i = 0; i < 32; ++i) o[i] = 0u;
  }
  const float l = __uint_as_float(lbits);
  const float inv_l = (n_ent > 0) ? 1.f / l : 0.f;
  if (row_valid) {
    if (p.out_fp32) {
      float4 *dst = reinterpret_cast<float4 *>(orow);
#pragma unroll
      for (int i = 0; i < 32; i += 4)
        dst[i >> 2] = make_float4(__uint_as_float(o[i]) * inv_l, __uint_as_float(o[i + 1]) * inv_l,
                                  __uint_as_float(o[i + 2]) * inv_l, __uint_as_float(o[i + 3]) * inv_l);
    } else {
      uint4 *dst = reinterpret_cast<uint4 *>(orow);
#pragma unroll
      for (int i = 0; i < 32; i += 8)
        dst[i >> 3] = make_uint4(pack_bf16x2(__uint_as_float(o[i]) * inv_l, __uint_as_float(o[i + 1]) * inv_l),
                                 pack_bf16x2(__uint_as_float(o[i + 2]) * inv_l, __uint_as_float(o[i + 3]) * inv_l),
                                 pack_bf16x2(__uint_as_float(o[i + 4]) * inv_l, __uint_as_float(o[i + 5]) * inv_l),
                                 pack_bf16x2(__uint_as_float(o[i + 6]) * inv_l, __uint_as_float(o[i + 7]) * inv_l));
    }
    if (!kFma && p.lse != nullptr)
      p.lse[(int64_t)h * p.N + tok] = (n_ent > 0) ? (m * c + log2f(l)) * 0.69314718055994531f : -INFINITY;
  }
}

// token-list mode: one warp gathers the B key (or value) rows of a tile into a SWIZZLE_128B stage with 16-byte cp.async copies
// (lane = 16-byte chunk (l & 7) of rows (l >> 3) + 4 i; padding rows are zero-filled); the stage's mbarrier (32 arrivals) completes
// when every lane's copies have landed.
template <int B>
__device__ __forceinline__ void gather_tile(const __nv_bfloat16 *__restrict__ base, int64_t stride_token, const int32_t *__restrict__ idx,
                                            int32_t n_kv, uint32_t stage, uint32_t bar_full) {
  const int lane = threadIdx.x & 31, ch = lane & 7, rr = lane >> 3;
#pragma unroll 8
  for (int it = 0; it < B / 4; ++it) {
    const int row = it * 4 + rr;
    const int j = __ldg(idx + row);
    const uint32_t dst = stage + row * 128 + ((ch ^ (row & 7)) << 4);
    const bool pad = j < 0 || j >= n_kv;  // -1 = padding; an index beyond the key tokens (a malformed caller-made list) is never dereferenced
    const __nv_bfloat16 *src = base + (int64_t)(pad ? 0 : j) * stride_token + ch * 8;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(pad ? 0 : 16) : "memory");
  }
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar_full) : "memory");
}

template <int B, bool kTok>
__global__ void __launch_bounds__(kAttnThreads, 2)
saf3r_attn_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                  const __grid_constant__ CUtensorMap map_v, const AttnParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  using L = AttnSmem<B>;
  const uint32_t sbase = smem_u32(smem);
  const int warp = threadIdx.x >> 5;
  const int I = blockIdx.x, h = p.head_order ? p.head_order[blockIdx.y] : (int)blockIdx.y;

  const uint32_t bar = sbase + L::kBar;
  const uint32_t bar_q = bar + 0;
  const uint32_t bar_k_full = bar + 8;                       // [kKStages]
  const uint32_t bar_k_empty = bar_k_full + 8 * kKStages;    // [kKStages]
  const uint32_t bar_v_full = bar_k_empty + 8 * kKStages;    // [kVStages]
  const uint32_t bar_v_empty = bar_v_full + 8 * kVStages;    // [kVStages]
  const uint32_t bar_s_full = bar_v_empty + 8 * kVStages;    // MMA -> softmax: S(e) is in TMEM
  const uint32_t bar_s_free = bar_s_full + 8;   // softmax -> MMA: S(e) has been read into registers (256 arrivals)
  const uint32_t bar_p_full = bar_s_free + 8;   // [2] softmax -> MMA: this 64-key half of P(e) is in TMEM, O rescaled (256 arrivals)
  const uint32_t bar_pv0_done = bar_p_full + 16;  // MMA -> softmax: the MMAs of the first half of P(e) are complete (P buffer free)
  const uint32_t bar_o_done = bar_pv0_done + 8;   // MMA -> softmax: PV(e) complete
  static_assert(8 + 16 * (kKStages + kVStages) + 48 <= 240, "barrier area overflow");
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::kBar + 248);
  constexpr int NH = B / 64;

  int64_t e0 = 0;
  int n_ent = p.NB_kv;
  if (kTok) {
    e0 = p.tile_ptr[I];
    const int64_t e1 = p.tile_ptr[I + 1];
    n_ent = (e0 < 0 || e1 < e0 || e1 > p.capacity_tiles) ? 0 : (int)(e1 - e0);  // out of the buffers: zero rows, lse = -inf
  } else if (p.row_ptr != nullptr) {
    const int64_t r = (int64_t)h * p.NB + I;
    e0 = p.row_ptr[r];
    n_ent = (int)(p.row_ptr[r + 1] - e0);
  }

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();  // SWIZZLE_128B tiles need a 1024-byte aligned base
    mbar_init(bar_q, 1);
    for (int s = 0; s < kKStages; ++s) { mbar_init(bar_k_full + 8 * s, kTok ? 32 : 1); mbar_init(bar_k_empty + 8 * s, 1); }
    for (int s = 0; s < kVStages; ++s) { mbar_init(bar_v_full + 8 * s, kTok ? 32 : 1); mbar_init(bar_v_empty + 8 * s, 1); }
    mbar_init(bar_s_full, 1);
    mbar_init(bar_s_free, 256);
    mbar_init(bar_p_full, 256);
    mbar_init(bar_p_full + 8, 256);
    mbar_init(bar_pv0_done, 1);
    mbar_init(bar_o_done, 1);
    fence_mbar_init();
  }
  // ones tile of the row-sum MMA: 16 rows x 64 bf16 of 1.0 (every 16-byte chunk is the same, so the 128-byte swizzle is a no-op)
  if (threadIdx.x >= 256) {
    reinterpret_cast<uint4 *>(smem + L::kOnes)[threadIdx.x - 256] = make_uint4(0x3f803f80u, 0x3f803f80u, 0x3f803f80u, 0x3f803f80u);
    fence_proxy_async_smem();
  }
  if (warp == 9) {
    tmem_alloc(smem_u32(tmem_slot), kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp >= 8) {
    setmaxnreg_dec<kRegsIdle>();
    if (warp == 8) {
      // ------------------------------------------------------------ TMA producer (warp-uniform loop, one elected lane issues)
      if (n_ent > 0) {
        if (elect_one_sync()) {
          tma_prefetch_desc(&map_q);
          tma_prefetch_desc(&map_k);
          tma_prefetch_desc(&map_v);
          mbar_arrive_expect_tx(bar_q, B * 128);
          tma_load_3d(sbase + L::kQ, &map_q, bar_q, 0, I * B, h);
        }
        __syncwarp();
        if (kTok) {  // warp 8 gathers the K tiles (warp 10 the V tiles, below)
          const __nv_bfloat16 *kb = p.k_base + (int64_t)h * p.kv_stride_head;
          int sk = 0, phk = 0;
          for (int e = 0; e < n_ent; ++e) {
            mbar_wait_relaxed<kSleepTma>(bar_k_empty + 8 * sk, phk ^ 1);
            gather_tile<B>(kb, p.kv_stride_token, p.key_idx + (e0 + e) * B, p.N_kv, sbase + L::kK + sk * B * 128, bar_k_full + 8 * sk);
            if (++sk == kKStages) { sk = 0; phk ^= 1; }
          }
        } else {
        int Jn = p.row_ptr ? p.col_idx[e0] : 0;
        int sk = 0, phk = 0, sv = 0, phv = 0;
        for (int e = 0; e < n_ent; ++e) {
          const int J = Jn;
          if (e + 1 < n_ent) Jn = p.row_ptr ? p.col_idx[e0 + e + 1] : e + 1;
          mbar_wait_relaxed<kSleepTma>(bar_k_empty + 8 * sk, phk ^ 1);
          if (elect_one_sync()) {
            mbar_arrive_expect_tx(bar_k_full + 8 * sk, B * 128);
            tma_load_3d(sbase + L::kK + sk * B * 128, &map_k, bar_k_full + 8 * sk, 0, J * B, h);
          }
          __syncwarp();
          mbar_wait_relaxed<kSleepTma>(bar_v_empty + 8 * sv, phv ^ 1);
          if (elect_one_sync()) {
            mbar_arrive_expect_tx(bar_v_full + 8 * sv, B * 128);
            tma_load_3d(sbase + L::kV + sv * B * 128, &map_v, bar_v_full + 8 * sv, 0, J * B, h);
          }
          __syncwarp();
          if (++sk == kKStages) { sk = 0; phk ^= 1; }
          if (++sv == kVStages) { sv = 0; phv ^= 1; }
        }
        }
      }
    } else if (kTok && warp == 10) {
      // ------------------------------------------------------------ token-list mode: gather producer of the V tiles
      const __nv_bfloat16 *vb = p.v_base + (int64_t)h * p.kv_stride_head;
      int sv = 0, phv = 0;
      for (int e = 0; e < n_ent; ++e) {
        mbar_wait_relaxed<kSleepTma>(bar_v_empty + 8 * sv, phv ^ 1);
        gather_tile<B>(vb, p.kv_stride_token, p.key_idx + (e0 + e) * B, p.N_kv, sbase + L::kV + sv * B * 128, bar_v_full + 8 * sv);
        if (++sv == kVStages) { sv = 0; phv ^= 1; }
      }
    } else if (warp == 9) {
      // ------------------------------------------------------------ MMA issuer (warp-uniform loop, one elected lane issues)
      if (n_ent > 0) {
        constexpr uint32_t idesc_qk = umma_idesc_bf16(B, false);
        constexpr uint32_t idesc_pv = umma_idesc_bf16(kD, true);
        const uint64_t qdesc = umma_desc_sw128(sbase + L::kQ);
        const uint32_t tS = tmem, tO = tmem + kTmemO, tP = tmem + kTmemP;
        int sk = 0, phk = 0;
        auto issue_qk = [&]() {
          mbar_wait_relaxed<kSleepMma>(bar_k_full + 8 * sk, phk);
          if (kTok) fence_proxy_async_smem();  // the gathered tile was written through the generic proxy (cp.async)
          tc_fence_after();
          if (elect_one_sync()) {
            const uint64_t kdesc = umma_desc_sw128(sbase + L::kK + sk * B * 128);
#pragma unroll
            for (int k = 0; k < kD / 16; ++k) umma_ss(tS, qdesc + 2 * k, kdesc + 2 * k, idesc_qk, k > 0);
            umma_commit(bar_k_empty + 8 * sk);
            umma_commit(bar_s_full);
          }
          __syncwarp();
          if (++sk == kKStages) { sk = 0; phk ^= 1; }
        };
        mbar_wait_relaxed<kSleepMma>(bar_q, 0);
        issue_qk();
        int sv = 0, phv = 0;
        constexpr uint32_t idesc_l = umma_idesc_bf16(16, false);
        const uint64_t odesc = umma_desc_sw128(sbase + L::kOnes);
        const uint32_t tL = tmem + kTmemL;
        for (int e = 0; e < n_ent; ++e) {
          if (e + 1 < n_ent) {
            mbar_wait_relaxed<kSleepMma>(bar_s_free, e & 1);  // S(e) is in registers -> overwrite it with S(e+1) while softmax(e) runs
            issue_qk();
          }
          mbar_wait_relaxed<kSleepMma>(bar_v_full + 8 * sv, phv);
          if (kTok) fence_proxy_async_smem();
#pragma unroll
          for (int hh = 0; hh < NH; ++hh) {
            mbar_wait_relaxed<kSleepMma>(bar_p_full + 8 * hh, e & 1);
            tc_fence_after();
            if (elect_one_sync()) {
              const uint64_t vdesc = umma_desc_sw128(sbase + L::kV + sv * B * 128);
#pragma unroll
              for (int kk = 0; kk < 4; ++kk)   // O += P_half . V_half (K = 16 keys per MMA; P packed: 8 columns per step)
                umma_ts(tO, (hh == 1 && kk < 2) ? tmem + kTmemPB + kk * 8 : tP + kk * 8, vdesc + (uint64_t)(hh * 4 + kk) * 128, idesc_pv, (e > 0 || hh > 0 || kk > 0) ? 1u : 0u);
#pragma unroll
              for (int kk = 0; kk < 4; ++kk)   // l += P_half . 1 (N = 16 identical columns)
                umma_ts(tL, (hh == 1 && kk < 2) ? tmem + kTmemPB + kk * 8 : tP + kk * 8, odesc + 2 * kk, idesc_l, (e > 0 || hh > 0 || kk > 0) ? 1u : 0u);
              if (hh + 1 < NH) {
                umma_commit(bar_pv0_done);
              } else {
                umma_commit(bar_v_empty + 8 * sv);
                umma_commit(bar_o_done);
              }
            }
            __syncwarp();
          }
          if (++sv == kVStages) { sv = 0; phv ^= 1; }
        }
      }
    }
  } else if (warp < 4) {
    setmaxnreg_inc<kRegsMufu>();
    softmax_half<B, false, kTok>(p, smem, tmem, n_ent, e0, h, I, bar_q, bar_s_full, bar_s_free, bar_p_full, bar_pv0_done, bar_o_done);
  } else {
    setmaxnreg_inc<kRegsFma>();
    softmax_half<B, true, kTok>(p, smem, tmem, n_ent, e0, h, I, bar_q, bar_s_full, bar_s_free, bar_p_full, bar_pv0_done, bar_o_done);
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 9) {
    __syncwarp();
    tmem_dealloc(tmem, kTmemCols);
  }
}

// kmax[h] = max over the head's key tokens of |k_j|_2 (the Cauchy-Schwarz factor of the freeze test above).  One streaming pass
// over K: grid (chunks, H), 256 threads, 8 lanes per 128-byte token row with eight 16-byte loads in flight per lane; the norms
// are non-negative, so the maximum of their bit patterns as unsigned integers is the maximum of the floats (atomicMax into a
// zeroed slot).  Thread 0 of CTA (0, 0) also writes the head order of the attention launch.
constexpr int kKnormRows = 1024;  // token rows per CTA
__global__ void __launch_bounds__(256) knorm_kernel(const __nv_bfloat16 *__restrict__ k, int64_t n_kv, int64_t stride_head,
                                                    int64_t stride_token, float *__restrict__ kmax, const int64_t *__restrict__ row_ptr,
                                                    int NB, uint8_t *__restrict__ head_order) {
  const int h = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
    // scheduling aid for the attention launch that follows: heads by total list length, longest first (stable insertion sort of
    // at most SAF3R_MAX_HEADS entries; dense mode / token lists: identity)
    const int H = gridDim.y;
    int64_t len[SAF3R_MAX_HEADS];
    uint8_t ord[SAF3R_MAX_HEADS];
    for (int i = 0; i < H; ++i) {
      len[i] = row_ptr ? row_ptr[(int64_t)(i + 1) * NB] - row_ptr[(int64_t)i * NB] : 0;
      ord[i] = (uint8_t)i;
    }
    for (int a = 1; a < H; ++a)
      for (int b = a; b > 0 && len[ord[b - 1]] < len[ord[b]]; --b) {
        const uint8_t t = ord[b];
        ord[b] = ord[b - 1];
        ord[b - 1] = t;
      }
    for (int i = 0; i < H; ++i) head_order[i] = ord[i];
  }
  const int sub = lane & 7, rg = lane >> 3;
  const int64_t t0 = (int64_t)blockIdx.x * kKnormRows + warp * (kKnormRows / 8);
  const __nv_bfloat16 *src = k + (int64_t)h * stride_head + sub * 8;
  float best = 0.f;
#pragma unroll 1
  for (int r0 = 0; r0 < kKnormRows / 8; r0 += 32) {
    uint4 raw[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int64_t t = t0 + r0 + rg + 4 * i;
      raw[i] = make_uint4(0, 0, 0, 0);
      if (t < n_kv) asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(raw[i].x), "=r"(raw[i].y), "=r"(raw[i].z), "=r"(raw[i].w) : "l"(src + t * stride_token));
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const uint32_t u[4] = {raw[i].x, raw[i].y, raw[i].z, raw[i].w};
      float ss = 0.f;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const float lo = __uint_as_float(u[c] << 16), hi = __uint_as_float(u[c] & 0xffff0000u);
        ss = fmaf(lo, lo, ss);
        ss = fmaf(hi, hi, ss);
      }
      ss += __shfl_xor_sync(0xffffffffu, ss, 1);
      ss += __shfl_xor_sync(0xffffffffu, ss, 2);
      ss += __shfl_xor_sync(0xffffffffu, ss, 4);
      best = fmaxf(best, ss);
    }
  }
#pragma unroll
  for (int off = 8; off < 32; off <<= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, off));
  __shared__ float wmax[8];
  if (lane == 0) wmax[warp] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    float b = wmax[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) b = fmaxf(b, wmax[w]);
    atomicMax(reinterpret_cast<unsigned int *>(kmax + h), __float_as_uint(sqrtf(b) * 1.0001f));
  }
}

}  // namespace saf3r
