// kernels_router_tc.cuh — router logits (a1, first half) on the 5th-gen tensor cores.
//
// logits[t, e] = sum_h x[t, h] * W_r[e, h]   ("A learned gating mechanism")
//
// The expert indices must match an fp64 oracle outside near-ties of 1e-4 (north_star), so the
// fp32 router weights cannot simply be rounded to bf16 or TF32 (SURVEY.md §7 hard part 4: that
// flips memberships well outside the allowance).  x is already exact bf16, so W_r is split once
// at create into two bf16 terms  W_r = hi + lo + O(2^-17 |W_r|)  and the kernel issues two
// kind::f16 MMAs per K step into the same fp32 TMEM accumulator.  Products are exact, the
// accumulation is the tensor core's fp32; the logit error stays near 1e-5 (measured in the parity
// tests through the SLP_BUF_LOGITS export), a decade below the near-tie allowance.
//
//   grid   (ceil(T / (128 kRowTiles)), ceil(E / 256)); kRowTiles 128-token x <=256-expert tiles per CTA.  Every CTA
//          streams the whole split W_r (7.3 MB for 256 x 7168) through its shared memory, so with one row tile per
//          CTA the kernel is bound by L2 -> SM traffic (2.35 GB through the crossbar for 0.48 GB of DRAM at 32K
//          tokens); two row tiles per CTA (two fp32 accumulators = all 512 TMEM columns) halve it.  The host picks
//          kRowTiles = 2 when one row tile per CTA would need more than one wave of CTAs.
//   warp 4 TMA producer: kRowTiles x tiles (128 rows x 64 bf16) + hi and lo tiles of W_r per K step,
//          128B-swizzled 2-stage ring
//   warp 5 MMA issuer: 4 K sub-steps x {hi, lo} tcgen05.mma.kind::f16 (M128, N = tile experts)
//   warps 0-3 epilogue: tcgen05.ld -> fp32 logits rows
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_bf16.h>
#include "ptx.cuh"

namespace slp {
namespace rtc {

constexpr int BM = 128, BKB = 128 /* bytes of K per step = 64 bf16 */, BN = 256;
constexpr int kStages = 2;
constexpr int kABytes = BM * BKB, kBoxBytes = 128 * BKB;
constexpr int kThreads = 192;
template <int kRowTiles> struct Cfg {
  static constexpr int kStageBytes = kRowTiles * kABytes + 4 * kBoxBytes;  // A tiles | hi (2 boxes) | lo (2 boxes)
  static constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 128 /*barriers*/;
  static_assert(kSmemBytes <= 232448, "shared memory budget");
};

// W_r [E, H] fp32 -> hl [2][Erows][H] bf16 bit patterns (hi, then lo = bf16(w - hi)); rows >= E stay 0.
__global__ void __launch_bounds__(256) split_router_w_kernel(const float* __restrict__ w, uint16_t* __restrict__ hl, int E, int H,
                                                             int Erows) {
  const size_t n = static_cast<size_t>(E) * H;
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < n; i += static_cast<size_t>(gridDim.x) * blockDim.x) {
    const float v = w[i];
    const __nv_bfloat16 hi = __float2bfloat16_rn(v);
    const __nv_bfloat16 lo = __float2bfloat16_rn(v - __bfloat162float(hi));
    hl[i] = *reinterpret_cast<const uint16_t*>(&hi);
    hl[static_cast<size_t>(Erows) * H + i] = *reinterpret_cast<const uint16_t*>(&lo);
  }
}

struct Shared {
  uint64_t full[kStages];
  uint64_t empty[kStages];
  uint64_t tmem_full;
  uint32_t tmem_base;
  int dead;
};

// tm_x: hidden viewed as uint8 [T, 2H]; tm_w: hl viewed as uint8 [2 * Erows, 2H]; both with
// 128 B x 128 row boxes and 128B swizzle (rows past the end are zero-filled by TMA).
template <int kRowTiles>
__global__ void __launch_bounds__(kThreads, 1)
router_logits_tc_kernel(const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_w,
                        float* __restrict__ logits, int T, int H, int E, int Erows, int* err) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  constexpr int kStageBytes = Cfg<kRowTiles>::kStageBytes, kWOff = kRowTiles * kABytes;
  constexpr int kTmemCols = kRowTiles * BN;
  Shared* sh = reinterpret_cast<Shared*>(smem + kStages * kStageBytes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.x * (kRowTiles * BM), n0 = blockIdx.y * BN;
  const int row_tiles = min(kRowTiles, (T - m0 + BM - 1) / BM);  // a last CTA may have one
  const int Nt = min(BN, (E - n0 + 15) / 16 * 16);  // MMA N: multiple of 16
  const int nbox = (Nt + 127) / 128;
  const int num_kb = (2 * H) / BKB;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&sh->full[i], 1); ptx::mbar_init(&sh->empty[i], 1); }
    ptx::mbar_init(&sh->tmem_full, 1);
    sh->dead = 0;
    ptx::fence_mbar_init();
  }
  if (warp == 5) ptx::tmem_alloc<kTmemCols>(&sh->tmem_base);
  if (warp == 4 && lane == 0) { ptx::prefetch_tmap(&tm_x); ptx::prefetch_tmap(&tm_w); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = sh->tmem_base;
  volatile int* dead = &sh->dead;

  if (warp == 4) {
    int stage = 0;
    uint32_t phase = 0;
    for (int kb = 0; kb < num_kb; ++kb) {
      ptx::mbar_wait(&sh->empty[stage], phase ^ 1, dead, err, 11);
      if (ptx::elect_one()) {
        uint8_t* sa = smem + stage * kStageBytes;
        uint8_t* sb = sa + kWOff;
        ptx::mbar_arrive_expect_tx(&sh->full[stage], row_tiles * kABytes + 2 * nbox * kBoxBytes);
        for (int rt = 0; rt < row_tiles; ++rt) ptx::tma_load_2d(sa + rt * kABytes, &tm_x, &sh->full[stage], kb * BKB, m0 + rt * BM);
        for (int b = 0; b < nbox; ++b) {
          ptx::tma_load_2d(sb + b * kBoxBytes, &tm_w, &sh->full[stage], kb * BKB, n0 + b * 128);
          ptx::tma_load_2d(sb + (2 + b) * kBoxBytes, &tm_w, &sh->full[stage], kb * BKB, Erows + n0 + b * 128);
        }
      }
      __syncwarp();
      if (++stage == kStages) { stage = 0; phase ^= 1; }
    }
  } else if (warp == 5) {
    const uint32_t idesc = ptx::umma_idesc_bf16_f32(BM, Nt);
    int stage = 0;
    uint32_t phase = 0;
    for (int kb = 0; kb < num_kb; ++kb) {
      ptx::mbar_wait(&sh->full[stage], phase, dead, err, 12);
      ptx::tc_fence_after();
      if (ptx::elect_one()) {
        const uint8_t* sa = smem + stage * kStageBytes;
        const uint64_t hdesc = ptx::umma_desc_k128(sa + kWOff);
        const uint64_t ldesc = ptx::umma_desc_k128(sa + kWOff + 2 * kBoxBytes);
        for (int rt = 0; rt < row_tiles; ++rt) {
          const uint64_t adesc = ptx::umma_desc_k128(sa + rt * kABytes);
#pragma unroll
          for (int k4 = 0; k4 < BKB / 32; ++k4) {  // UMMA_K = 16 bf16 = 32 B per step
            ptx::umma_bf16(tmem_base + rt * BN, adesc + 2 * k4, hdesc + 2 * k4, idesc, (kb | k4) > 0);
            ptx::umma_bf16(tmem_base + rt * BN, adesc + 2 * k4, ldesc + 2 * k4, idesc, 1);
          }
        }
        ptx::umma_commit(&sh->empty[stage]);
        if (kb == num_kb - 1) ptx::umma_commit(&sh->tmem_full);
      }
      __syncwarp();
      if (++stage == kStages) { stage = 0; phase ^= 1; }
    }
  } else {
    ptx::mbar_wait(&sh->tmem_full, 0, dead, err, 13);
    ptx::tc_fence_after();
   for (int rt = 0; rt < row_tiles; ++rt) {
    const int t = m0 + rt * BM + warp * 32 + lane;
    const uint32_t tb = tmem_base + (static_cast<uint32_t>(warp * 32) << 16) + rt * BN;
    for (int c = 0; c < Nt; c += 16) {
      uint32_t v[16];
      ptx::tmem_ld16(tb + c, v);
      ptx::tmem_ld_wait16(v);
      if (t < T) {
        float* dst = logits + static_cast<size_t>(t) * E + n0 + c;
        if (n0 + c + 16 <= E && (E & 3) == 0) {
#pragma unroll
          for (int i = 0; i < 4; ++i)
            reinterpret_cast<float4*>(dst)[i] = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]),
                                                            __uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3]));
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (n0 + c + i < E) dst[i] = __uint_as_float(v[i]);
        }
      }
    }
   }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 5) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<kTmemCols>(tmem_base);
  }
}

}  // namespace rtc
}  // namespace slp
