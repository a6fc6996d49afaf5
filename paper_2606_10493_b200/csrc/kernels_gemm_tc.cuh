// kernels_gemm_tc.cuh — grouped FP8 GEMM on the 5th-gen tensor cores (a5, a6, a7, a8).
//
// One persistent CTA per SM walks a static round-robin list of (128-row tile, N tile) pairs over
// the experts of the launch.  Per 128-deep K block the tensor core writes a fresh 128 x 256 fp32
// partial into TMEM; the promotion warps pull it out with tcgen05.ld and add it into fp32 register
// accumulators with one FMA per element, scaled by  xs[row, kb] * ws[n-block, kb]
// ("FP8 GEMM with FP32 accumulation"; "accumulate all partial
// dot-products first and apply the scale once per block").
//
// The 256 accumulator columns of a K block are produced as two independent 128-column halves,
// each with its own TMEM full/empty barrier pair and its own group of four promotion warps, and
// TMEM holds two K blocks (4 half buffers).  Promotion of a half needs ~380 cycles of the ~512 a
// K block takes on the tensor core, so the hand-off latencies only hide if a half can be refilled
// three half-slots (768 cycles) after it was published (measured: profiles/r1_*).
//
//   warp 8      TMA producer: A tile (128 rows x 128 B) + four 64-row B boxes per K block into a
//               4-stage 128B-swizzled smem ring (mbarrier full/empty)
//   warp 9      MMA issuer: per K block and half, 4 x tcgen05.mma.kind::f8f6f4 (M128 N128 K32)
//               into TMEM columns buf * 256 + half * 128; tcgen05.commit publishes the half and
//               (after the second half) frees the smem stage
//   warps 10-11 idle (they only donate their registers, setmaxnreg)
//   warps 0-7   promotion + epilogue: warp w owns TMEM lanes 32 * (w % 4).. (rows) of half w / 4;
//               128 fp32 accumulators per thread
//
// kMode 0 (gate/up): B smem rows = [gate n0..+63 | up n0..+63 | gate n0+64..+127 | up n0+64..+127],
//   so each half holds the gate and up columns of the same 64 intermediate channels; epilogue
//   h = silu(g) * u, row amax over the 128 channels (two halves, exchanged through smem),
//   s = amax / 448, e4m3(h / s) -> hq, hs  ("SiLU(.) (.)"; Q14).
// kMode 1 (down):   B = down rows n0..n0+255; epilogue fp32 store of Y through a per-warp smem
//   transpose so that every store instruction writes whole 128-byte lines (Y stays fp32 so that
//   the only bf16 rounding of the layer is the final one in the combine).
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include "ptx.cuh"
#include "kernels_gemm_simt.cuh"  // GemmArgs, slot_of, rows_of

namespace slp {
namespace tc {

constexpr int BM = 128, BN = 256, BK = 128, HN = 128;
constexpr int kStages = 4;
constexpr int kABytes = BM * BK, kBBytes = BN * BK, kStageBytes = kABytes + kBBytes;
constexpr int kBoxRows = 64;  // rows per B TMA box
#ifndef SLP_SPLIT_N
#define SLP_SPLIT_N 0
#endif
constexpr bool kSplitN = SLP_SPLIT_N;  // issue each K block as two N = 128 MMA groups (finer TMEM hand-off, but A is read twice from smem)
constexpr int kEpiWarps = 8;
constexpr int kThreads = (kEpiWarps + 4) * 32;  // three warpgroups: 2 x promotion, 1 x {producer, MMA, 2 idle}
constexpr int kTmemCols = 512;
constexpr int kScratchBytes = kEpiWarps * 32 * 32 * 4;  // per-warp 32 x 32 fp32 transpose tile (mode 1) / amax exchange (mode 0)
constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 256 /*barriers*/ + kScratchBytes;

struct Shared {
  uint64_t full[kStages];
  uint64_t empty[kStages];
  uint64_t tmem_full[4];   // [buf * 2 + half]
  uint64_t tmem_empty[4];
  uint32_t tmem_base;
  int dead;
};
static_assert(sizeof(Shared) <= 256, "barrier block");

// silu(g) * u with the fast exponential and reciprocal (rel. error ~1e-6, three decades below the
// e4m3 step that follows).
__device__ __forceinline__ float silu_mul_fast(float g, float u) { return __fdividef(g, 1.0f + __expf(-g)) * u; }

// Correctly rounded h / s from a correctly rounded reciprocal and one residual step (Markstein):
// q0 = h * r, q = q0 + (h - q0 * s) * r.
__device__ __forceinline__ float div_by(float h, float s, float r) {
  const float q0 = h * r;
  return fmaf(fmaf(-q0, s, h), r, q0);
}
__device__ __forceinline__ uint32_t quant4_e4m3_r(float a, float b, float c, float d, float s, float r) {
  __nv_fp8x2_storage_t lo = __nv_cvt_float2_to_fp8x2(make_float2(div_by(a, s, r), div_by(b, s, r)), __NV_SATFINITE, __NV_E4M3);
  __nv_fp8x2_storage_t hi = __nv_cvt_float2_to_fp8x2(make_float2(div_by(c, s, r), div_by(d, s, r)), __NV_SATFINITE, __NV_E4M3);
  return static_cast<uint32_t>(lo) | (static_cast<uint32_t>(hi) << 16);
}

template <int kMode>
__global__ void __launch_bounds__(kThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b, GemmArgs g) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  Shared* sh = reinterpret_cast<Shared*>(smem + kStages * kStageBytes);
  uint8_t* scratch = smem + kStages * kStageBytes + 256;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K = kMode == 0 ? g.H : g.I;
  const int N = kMode == 0 ? g.I : g.H;
  const int num_kb = K / BK;
  const int n_tiles = kMode == 0 ? N / 128 : (N + BN - 1) / BN;
  const int mt_begin = g.tile_start[g.e_begin], mt_end = g.tile_start[g.e_end];
  const int total = (mt_end - mt_begin) * n_tiles;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&sh->full[i], 1); ptx::mbar_init(&sh->empty[i], 1); }
    for (int i = 0; i < 4; ++i) { ptx::mbar_init(&sh->tmem_full[i], 1); ptx::mbar_init(&sh->tmem_empty[i], kEpiWarps / 2); }
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

  // Work item w -> (m tile, n tile): n fastest, so the CTAs running together cover a few m tiles
  // of one expert against all of its N tiles and share both operands through L2.
  auto decode = [&](int w, int& mt, int& nt) {
    mt = mt_begin + w / n_tiles;
    nt = w % n_tiles;
  };

  // Registers: 168 per thread at launch (384 threads); the producer / MMA warpgroup gives most of
  // its share to the two promotion warpgroups, which hold 128 accumulators + two loads in flight.
  if (warp >= kEpiWarps) {
   ptx::setmaxnreg_dec<40>();
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
      int brow[4];
      if (kMode == 0) {
        const int gate0 = slot * 3 * g.I + nt * 128;  // view [slots*3I, H]
        brow[0] = gate0; brow[1] = gate0 + g.I; brow[2] = gate0 + 64; brow[3] = gate0 + g.I + 64;
      } else {
        const int down0 = slot * 3 * g.H + 2 * g.H + nt * BN;  // view [slots*3H, I]
        brow[0] = down0; brow[1] = down0 + 64; brow[2] = down0 + 128; brow[3] = down0 + 192;
      }
      for (int kb = 0; kb < num_kb; ++kb) {
        ptx::mbar_wait(&sh->empty[stage], phase ^ 1, dead, g.err, 1);
        if (ptx::elect_one()) {
          uint8_t* sa = smem + stage * kStageBytes;
          uint8_t* sb = sa + kABytes;
          ptx::mbar_arrive_expect_tx(&sh->full[stage], kStageBytes);
          ptx::tma_load_2d(sa, &tm_a, &sh->full[stage], kb * BK, row0);
#pragma unroll
          for (int b = 0; b < 4; ++b) ptx::tma_load_2d(sb + b * kBoxRows * BK, &tm_b, &sh->full[stage], kb * BK, brow[b]);
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == kEpiWarps + 1) {
    // ===================== MMA issuer =====================
    constexpr uint32_t idesc_half = ptx::umma_idesc_e4m3_f32(BM, HN), idesc_full = ptx::umma_idesc_e4m3_f32(BM, BN);
    int stage = 0;
    uint32_t phase = 0;
    uint32_t it = 0;  // running K-block counter: TMEM buffer = it & 1
    for (int w = blockIdx.x; w < total; w += gridDim.x) {
      for (int kb = 0; kb < num_kb; ++kb, ++it) {
        const uint32_t buf = it & 1, tph = ((it >> 1) & 1) ^ 1;
        ptx::mbar_wait(&sh->full[stage], phase, dead, g.err, 3);
        if (kSplitN) {
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            ptx::mbar_wait(&sh->tmem_empty[buf * 2 + half], tph, dead, g.err, 2);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
              const uint8_t* sa = smem + stage * kStageBytes;
              const uint64_t adesc = ptx::umma_desc_k128(sa);
              const uint64_t bdesc = ptx::umma_desc_k128(sa + kABytes + half * HN * BK);
              const uint32_t d = tmem_base + buf * BN + half * HN;
#pragma unroll
              for (int k4 = 0; k4 < BK / 32; ++k4)  // UMMA_K = 32 for 8-bit operands: +32 B per step
                ptx::umma_f8(d, adesc + 2 * k4, bdesc + 2 * k4, idesc_half, k4 > 0);
              if (half == 1) ptx::umma_commit(&sh->empty[stage]);   // smem stage reusable once these MMAs retire
              ptx::umma_commit(&sh->tmem_full[buf * 2 + half]);     // this half of the K block's partial is complete
            }
            __syncwarp();
          }
        } else {
          ptx::mbar_wait(&sh->tmem_empty[buf * 2], tph, dead, g.err, 2);
          ptx::mbar_wait(&sh->tmem_empty[buf * 2 + 1], tph, dead, g.err, 2);
          ptx::tc_fence_after();
          if (ptx::elect_one()) {
            const uint8_t* sa = smem + stage * kStageBytes;
            const uint64_t adesc = ptx::umma_desc_k128(sa);
            const uint64_t bdesc = ptx::umma_desc_k128(sa + kABytes);
            const uint32_t d = tmem_base + buf * BN;
#pragma unroll
            for (int k4 = 0; k4 < BK / 32; ++k4) ptx::umma_f8(d, adesc + 2 * k4, bdesc + 2 * k4, idesc_full, k4 > 0);
            ptx::umma_commit(&sh->empty[stage]);
            ptx::umma_commit(&sh->tmem_full[buf * 2]);
            ptx::umma_commit(&sh->tmem_full[buf * 2 + 1]);
          }
          __syncwarp();
        }
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
   }
  } else {
    // ===================== promotion + epilogue =====================
    ptx::setmaxnreg_inc<232>();
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
      const float* as_ptr = g.a_s + row * g.a_s_stride;  // padded to a multiple of 4 floats, 16-byte aligned
      // weight-scale rows of this thread's columns: chunks 0-3 use ws0, chunks 4-7 use ws1
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

      // Scales are fetched far ahead of use: the row's activation scales four K blocks at a time
      // (one 16-byte load), the weight scales 32 K blocks at a time, one per lane, broadcast by shuffle.
      float4 xs_nxt = row_ok ? *reinterpret_cast<const float4*>(as_ptr) : make_float4(0.f, 0.f, 0.f, 0.f);
      float w0_nxt = lane < num_kb ? ws0[lane] : 0.f, w1_nxt = lane < num_kb ? ws1[lane] : 0.f;
      float w0_cur = 0.f, w1_cur = 0.f;
      for (int kb4 = 0; kb4 < num_kb; kb4 += 4) {
        const float4 xs_cur = xs_nxt;
        if (kb4 + 4 < num_kb && row_ok) xs_nxt = *reinterpret_cast<const float4*>(as_ptr + kb4 + 4);
        if ((kb4 & 31) == 0) {
          w0_cur = w0_nxt;
          w1_cur = w1_nxt;
          const int kn = kb4 + 32 + lane;
          w0_nxt = kn < num_kb ? ws0[kn] : 0.f;
          w1_nxt = kn < num_kb ? ws1[kn] : 0.f;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int kb = kb4 + j;
          if (kb >= num_kb) break;
          const float sa = j == 0 ? xs_cur.x : j == 1 ? xs_cur.y : j == 2 ? xs_cur.z : xs_cur.w;
          const float sc0 = sa * __shfl_sync(0xFFFFFFFFu, w0_cur, kb & 31);
          const float sc1 = kMode == 0 ? sa * __shfl_sync(0xFFFFFFFFu, w1_cur, kb & 31) : sc0;
          const uint32_t buf = it & 1;
          ptx::mbar_wait(&sh->tmem_full[buf * 2 + half], (it >> 1) & 1, dead, g.err, 4);
          ptx::tc_fence_after();
          const uint32_t tb = tmem_base + lane_addr + buf * BN + half * HN;
          // 8 chunks of 16 columns, two register sets in flight
          uint32_t v0[16], v1[16];
          ptx::tmem_ld16(tb, v0);
#pragma unroll
          for (int c = 0; c < 8; c += 2) {
            ptx::tmem_ld_wait16(v0);
            ptx::tmem_ld16(tb + (c + 1) * 16, v1);
            ptx::keep16(v0);  // v0 stays live across the issue of the next load: distinct registers
            {
              const float sc = (c < 4) ? sc0 : sc1;
#pragma unroll
              for (int i = 0; i < 16; ++i) acc[c * 16 + i] = fmaf(__uint_as_float(v0[i]), sc, acc[c * 16 + i]);
            }
            ptx::tmem_ld_wait16(v1);
            if (c + 2 < 8) {
              ptx::tmem_ld16(tb + (c + 2) * 16, v0);
              ptx::keep16(v1);
            }
            {
              const float sc = (c + 1 < 4) ? sc0 : sc1;
#pragma unroll
              for (int i = 0; i < 16; ++i) acc[(c + 1) * 16 + i] = fmaf(__uint_as_float(v1[i]), sc, acc[(c + 1) * 16 + i]);
            }
          }
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(&sh->tmem_empty[buf * 2 + half]);
          ++it;
        }
      }

      if (kMode == 0) {
        // h = silu(gate) * up over this thread's 64 channels; row amax over all 128 via smem
        float amax = 0.f;
#pragma unroll
        for (int i = 0; i < 64; ++i) {
          acc[i] = silu_mul_fast(acc[i], acc[64 + i]);
          amax = fmaxf(amax, fabsf(acc[i]));
        }
        float* ex = reinterpret_cast<float*>(scratch) + tile_parity * 2 * BM;  // [parity][half][row]
        ex[half * BM + r_in_tile] = amax;
        ptx::named_bar_sync(1, kEpiWarps * 32);
        amax = fmaxf(amax, ex[(half ^ 1) * BM + r_in_tile]);
        const float s = (amax == 0.f) ? 1.0f : __fdiv_rn(amax, 448.0f);
        if (row_ok) {
          uint32_t pk[16];
          if (s > 1e-30f) {
            const float r = __frcp_rn(s);
#pragma unroll
            for (int i = 0; i < 16; ++i) pk[i] = quant4_e4m3_r(acc[4 * i], acc[4 * i + 1], acc[4 * i + 2], acc[4 * i + 3], s, r);
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) pk[i] = quant4_e4m3(acc[4 * i], acc[4 * i + 1], acc[4 * i + 2], acc[4 * i + 3], s);
          }
          uint4* dst = reinterpret_cast<uint4*>(g.hq + row * g.I + nt * 128 + half * 64);
#pragma unroll
          for (int i = 0; i < 4; ++i) dst[i] = make_uint4(pk[4 * i], pk[4 * i + 1], pk[4 * i + 2], pk[4 * i + 3]);
          if (half == 0) g.hs[row * g.hs_stride + nt] = s;
        }
      } else {
        // Y tile: transpose 32 x 32 fp32 quarters through this warp's smem tile (16-byte chunks
        // XOR-swizzled by row) and store whole 128-byte row segments.
        const int c0 = nt * BN + half * HN;
        float4* st = reinterpret_cast<float4*>(scratch + warp * 4096);
        if (c0 < g.H) {
#pragma unroll
          for (int qq = 0; qq < 4; ++qq) {
#pragma unroll
            for (int j = 0; j < 8; ++j)
              st[lane * 8 + (j ^ (lane & 7))] = make_float4(acc[qq * 32 + j * 4], acc[qq * 32 + j * 4 + 1], acc[qq * 32 + j * 4 + 2], acc[qq * 32 + j * 4 + 3]);
            __syncwarp();
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int rr = i * 4 + (lane >> 3), jj = lane & 7;
              const float4 v = st[rr * 8 + (jj ^ (rr & 7))];
              if (q * 32 + rr < nrows)
                *reinterpret_cast<float4*>(g.y + static_cast<size_t>(row0 + q * 32 + rr) * g.H + c0 + qq * 32 + jj * 4) = v;
            }
            __syncwarp();
          }
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
