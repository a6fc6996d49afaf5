// kernels_gemm_tc.cuh — grouped FP8 GEMM on the 5th-gen tensor cores (a5, a6, a7, a8).
//
// One persistent CTA per SM walks a static round-robin list of (128-row tile, N tile) pairs over
// the experts of the launch.  Per 128-deep K block the tensor core writes a fresh 128 x 256 fp32
// partial into one of two TMEM buffers; the epilogue warps pull it out with tcgen05.ld and
// promote it into fp32 register accumulators with one FMA per element, scaled by
// xs[row, kb] * ws[n-block, kb]  ("FP8 GEMM with FP32 accumulation"; PAPER.md:255
// "accumulate all partial dot-products first and apply the scale once per block").
//
//   warp 8      TMA producer: A tile (128 rows x 128 B) + two B half-tiles (128 rows x 128 B each)
//               per K block into a 4-stage 128B-swizzled smem ring (mbarrier full/empty)
//   warp 9      MMA issuer: 4 x tcgen05.mma.kind::f8f6f4 (M128 N256 K32) per K block into TMEM
//               buffer kb % 2; tcgen05.commit frees the smem stage and publishes the buffer
//   warps 0-7   promotion + epilogue: warp w owns TMEM lanes 32*(w%4).. (rows) and half of the
//               columns (w/4); 128 fp32 accumulators per thread
//
// kMode 0 (gate/up): B = [gate rows n0..n0+127 | up rows n0..n0+127] of the expert; epilogue
//   h = silu(g) * u, row amax over the 128 channels, s = amax / 448, e4m3(h / s) -> hq, hs
//   ("SiLU(.) (.)"; fused requantisation, Q14).
// kMode 1 (down):   B = down rows n0..n0+255; epilogue fp32 store of Y (kept in fp32 so that the
//   only bf16 rounding of the layer is the final one in the combine).
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include "ptx.cuh"
#include "kernels_gemm_simt.cuh"  // GemmArgs, slot_of, rows_of, silu_mul

namespace slp {
namespace tc {

constexpr int BM = 128, BN = 256, BK = 128;
constexpr int kStages = 4;
constexpr int kABytes = BM * BK, kBBytes = BN * BK, kStageBytes = kABytes + kBBytes;
constexpr int kEpiWarps = 8;
constexpr int kThreads = (kEpiWarps + 2) * 32;
constexpr int kTmemCols = 512;
constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 256 /*barriers*/ + 2 * 2 * BM * 4 /*amax exchange*/;

struct Shared {
  uint64_t full[kStages];
  uint64_t empty[kStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint32_t tmem_base;
  int dead;
};

template <int kMode>
__global__ void __launch_bounds__(kThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b, GemmArgs g) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  Shared* sh = reinterpret_cast<Shared*>(smem + kStages * kStageBytes);
  float* amax_x = reinterpret_cast<float*>(smem + kStages * kStageBytes + 256);  // [2 parity][2 half][128 rows]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K = kMode == 0 ? g.H : g.I;
  const int N = kMode == 0 ? g.I : g.H;
  const int num_kb = K / BK;
  const int n_tiles = kMode == 0 ? N / 128 : (N + BN - 1) / BN;
  const int mt_begin = g.tile_start[g.e_begin], mt_end = g.tile_start[g.e_end];
  const int total = (mt_end - mt_begin) * n_tiles;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&sh->full[i], 1); ptx::mbar_init(&sh->empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&sh->tmem_full[i], 1); ptx::mbar_init(&sh->tmem_empty[i], kEpiWarps); }
    sh->dead = 0;
    ptx::fence_mbar_init();
  }
  if (warp == kEpiWarps + 1) ptx::tmem_alloc<kTmemCols>(&sh->tmem_base);
  if (warp == kEpiWarps && lane == 0) { ptx::prefetch_tmap(&tm_a); ptx::prefetch_tmap(&tm_b); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = sh->tmem_base;
  volatile int* dead = &sh->dead;

  // Work item w -> (m tile, n tile): m fastest, so CTAs running together share the B tile.
  auto decode = [&](int w, int& mt, int& nt) {
    // order: expert-major via mt ranges is implicit (tiles are sorted by expert); within the
    // launch walk n-tile-major over blocks of consecutive m tiles of one expert would need the
    // expert bounds; m fastest over the whole launch keeps A tiles hot instead when experts are
    // small.  Use n-major inside an expert: tiles of an expert are contiguous in mt.
    mt = mt_begin + w / n_tiles;
    nt = w % n_tiles;
  };

  if (warp == kEpiWarps) {
    // ===================== TMA producer =====================
    int stage = 0;
    uint32_t phase = 0;
    for (int w = blockIdx.x; w < total; w += gridDim.x) {
      int mt, nt;
      decode(w, mt, nt);
      const int e = g.tile_expert[mt];
      const int row0 = g.row_start[e] + (mt - g.tile_start[e]) * BM;
      const int slot = slot_of(g, e);
      int brow0, brow1;
      if (kMode == 0) {
        brow0 = slot * 3 * g.I + nt * 128;  // gate rows, view [slots*3I, H]
        brow1 = brow0 + g.I;                // up rows
      } else {
        brow0 = slot * 3 * g.H + 2 * g.H + nt * BN;  // down rows, view [slots*3H, I]
        brow1 = brow0 + 128;
      }
      for (int kb = 0; kb < num_kb; ++kb) {
        ptx::mbar_wait(&sh->empty[stage], phase ^ 1, dead, g.err, 1);
        if (lane == 0) {
          uint8_t* sa = smem + stage * kStageBytes;
          uint8_t* sb = sa + kABytes;
          ptx::mbar_arrive_expect_tx(&sh->full[stage], kStageBytes);
          ptx::tma_load_2d(sa, &tm_a, &sh->full[stage], kb * BK, row0);
          ptx::tma_load_2d(sb, &tm_b, &sh->full[stage], kb * BK, brow0);
          ptx::tma_load_2d(sb + 128 * BK, &tm_b, &sh->full[stage], kb * BK, brow1);
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == kEpiWarps + 1) {
    // ===================== MMA issuer =====================
    constexpr uint32_t idesc = ptx::umma_idesc_e4m3_f32(BM, BN);
    int stage = 0;
    uint32_t phase = 0;
    uint32_t it = 0;  // running K-block counter: TMEM buffer = it & 1
    for (int w = blockIdx.x; w < total; w += gridDim.x) {
      for (int kb = 0; kb < num_kb; ++kb, ++it) {
        const uint32_t buf = it & 1;
        ptx::mbar_wait(&sh->tmem_empty[buf], ((it >> 1) & 1) ^ 1, dead, g.err, 2);
        ptx::mbar_wait(&sh->full[stage], phase, dead, g.err, 3);
        ptx::tc_fence_after();
        if (lane == 0) {
          const uint8_t* sa = smem + stage * kStageBytes;
          const uint64_t adesc = ptx::umma_desc_k128(sa);
          const uint64_t bdesc = ptx::umma_desc_k128(sa + kABytes);
          const uint32_t d = tmem_base + buf * BN;
#pragma unroll
          for (int k4 = 0; k4 < BK / 32; ++k4)  // UMMA_K = 32 for 8-bit operands: +32 B per step
            ptx::umma_f8(d, adesc + 2 * k4, bdesc + 2 * k4, idesc, k4 > 0);
          ptx::umma_commit(&sh->empty[stage]);    // smem stage reusable once these MMAs retire
          ptx::umma_commit(&sh->tmem_full[buf]);  // partial of this K block complete
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  } else {
    // ===================== promotion + epilogue =====================
    const int q = warp & 3, half = warp >> 2;
    const int r_in_tile = q * 32 + lane;
    const uint32_t lane_addr = static_cast<uint32_t>(q * 32) << 16;
    uint32_t it = 0;
    int tile_parity = 0;
    for (int w = blockIdx.x; w < total; w += gridDim.x, tile_parity ^= 1) {
      int mt, nt;
      decode(w, mt, nt);
      const int e = g.tile_expert[mt];
      const int m_in_e = mt - g.tile_start[e];
      const int row0 = g.row_start[e] + m_in_e * BM;
      const int nrows = min(BM, rows_of(g, e) - m_in_e * BM);
      const size_t row = static_cast<size_t>(row0 + r_in_tile);
      const bool row_ok = r_in_tile < nrows;
      const float* as_ptr = g.a_s + row * g.a_s_stride;
      // weight-scale rows for this thread's two 64-column chunks groups
      const float *ws0, *ws1;
      if (kMode == 0) {
        const size_t o = (static_cast<size_t>(e) * (g.I / 128) + nt) * num_kb;
        ws0 = g.gate_s + o;
        ws1 = g.up_s + o;
      } else {
        const int nb = min(nt * 2 + half, g.H / 128 - 1);
        ws0 = g.down_s + (static_cast<size_t>(e) * (g.H / 128) + nb) * num_kb;
        ws1 = ws0;
      }
      float acc[128];
#pragma unroll
      for (int i = 0; i < 128; ++i) acc[i] = 0.f;

      float sa_n = row_ok ? as_ptr[0] : 0.f, w0_n = ws0[0], w1_n = ws1[0];
      for (int kb = 0; kb < num_kb; ++kb, ++it) {
        const float sc0 = sa_n * w0_n, sc1 = sa_n * w1_n;
        if (kb + 1 < num_kb) {  // prefetch next K block's scales
          sa_n = row_ok ? as_ptr[kb + 1] : 0.f;
          w0_n = ws0[kb + 1];
          w1_n = ws1[kb + 1];
        }
        const uint32_t buf = it & 1;
        ptx::mbar_wait(&sh->tmem_full[buf], (it >> 1) & 1, dead, g.err, 4);
        ptx::tc_fence_after();
        const uint32_t tb = tmem_base + lane_addr + buf * BN;
        // 8 chunks of 16 columns; chunk c lives at column col(c)
        auto col = [&](int c) -> uint32_t {
          return kMode == 0 ? (c < 4 ? half * 64 + c * 16 : 128 + half * 64 + (c - 4) * 16) : half * 128 + c * 16;
        };
        uint32_t v0[16], v1[16];
        ptx::tmem_ld16(tb + col(0), v0);
#pragma unroll
        for (int c = 0; c < 8; c += 2) {
          ptx::tmem_ld_wait16(v0);
          ptx::tmem_ld16(tb + col(c + 1), v1);
          {
            const float sc = (c < 4) ? sc0 : sc1;
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[c * 16 + i] = fmaf(__uint_as_float(v0[i]), sc, acc[c * 16 + i]);
          }
          ptx::tmem_ld_wait16(v1);
          if (c + 2 < 8) ptx::tmem_ld16(tb + col(c + 2), v0);
          {
            const float sc = (c + 1 < 4) ? sc0 : sc1;
#pragma unroll
            for (int i = 0; i < 16; ++i) acc[(c + 1) * 16 + i] = fmaf(__uint_as_float(v1[i]), sc, acc[(c + 1) * 16 + i]);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&sh->tmem_empty[buf]);
      }

      if (kMode == 0) {
        // h = silu(gate) * up over this thread's 64 channels; row amax over all 128 via smem
        float amax = 0.f;
#pragma unroll
        for (int i = 0; i < 64; ++i) {
          acc[i] = silu_mul(acc[i], acc[64 + i]);
          amax = fmaxf(amax, fabsf(acc[i]));
        }
        float* ex = amax_x + tile_parity * 2 * BM;
        ex[half * BM + r_in_tile] = amax;
        ptx::named_bar_sync(1, kEpiWarps * 32);
        amax = fmaxf(amax, ex[(half ^ 1) * BM + r_in_tile]);
        const float s = (amax == 0.f) ? 1.0f : __fdiv_rn(amax, 448.0f);
        if (row_ok) {
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) pk[i] = quant4_e4m3(acc[4 * i], acc[4 * i + 1], acc[4 * i + 2], acc[4 * i + 3], s);
          uint4* dst = reinterpret_cast<uint4*>(g.hq + row * g.I + nt * 128 + half * 64);
#pragma unroll
          for (int i = 0; i < 4; ++i) dst[i] = make_uint4(pk[4 * i], pk[4 * i + 1], pk[4 * i + 2], pk[4 * i + 3]);
          if (half == 0) g.hs[row * g.hs_stride + nt] = s;
        }
      } else {
        const int c0 = nt * BN + half * 128;
        if (row_ok && c0 < g.H) {
          float4* dst = reinterpret_cast<float4*>(g.y + row * g.H + c0);
#pragma unroll
          for (int i = 0; i < 32; ++i) dst[i] = make_float4(acc[4 * i], acc[4 * i + 1], acc[4 * i + 2], acc[4 * i + 3]);
        }
      }
    }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == kEpiWarps + 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<kTmemCols>(tmem_base);
  }
}

}  // namespace tc
}  // namespace slp
