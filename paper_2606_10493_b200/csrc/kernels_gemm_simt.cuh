// kernels_gemm_simt.cuh — plain CUDA-core grouped FP8 GEMM (triage "gemm=simt").
// Bring-up / triage scaffolding for the tcgen05 kernel in kernels_gemm_tc.cuh: same inputs, same
// outputs, same block-scale promotion structure (one fp32 partial per 128-deep K block, scaled by
// xs[row, kb] * ws[nb, kb] and added into an fp32 accumulator), but no tensor cores, no TMA.
#pragma once
#include <cstdint>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cuda_fp16.h>
#include "kernels_route.cuh"

namespace slp {

struct GemmArgs {
  // tile bookkeeping (written by permute_scan_kernel)
  const int32_t* tile_expert;  // [tiles] expert of each 128-row tile (E = shared)
  const int32_t* tile_start;   // [E+2]
  const int32_t* row_start;    // [E+2]
  const int32_t* counts;       // [E]
  const int4* tile_info;       // [tiles] {expert, first workspace row, valid rows, tile index inside the expert}
  const int32_t* pair_start;   // [E+2] prefix of ceil(m tiles / 2) per expert (CTA-pair GEMM work items)
  const int32_t* pair_expert;  // [pairs] expert of each pair of 128-row tiles
  int e_begin, e_end;          // experts covered by this launch: [e_begin, e_end), E = shared
  int E, T;
  int e_own0;                  // first routed expert this handle owns (SmallEP expert sharding; 0 on one GPU)
  int shared_rows;             // rows of the shared expert's token range (T on one GPU)
  int n_stage;                 // slot of routed expert e is 1 + (e - e_own0) % n_stage; shared expert: slot 0
  int n_slots;                 // 1 + n_stage slots per weight kind: pool = [gate slots | up slots | down slots]
  // operands
  const uint8_t* a_q;          // [rows, K] e4m3
  const float* a_s;            // [rows, a_s_stride]
  int a_s_stride;
  const uint8_t* pool;         // [3][n_slots][I*H]: gate [I,H] of every slot, then up [I,H], then down [H,I]
  const float* gate_s;         // [E+1, I/128, H/128]
  const float* up_s;           // [E+1, I/128, H/128]
  const float* down_s;         // [E+1, H/128, I/128]
  int H, I;
  // outputs
  uint8_t* hq;                 // [rows, I]
  float* hs;                   // [rows, hs_stride]
  int hs_stride;
  uint16_t* y;                 // [rows, H] fp16 bit patterns, block-scaled: value = y * ys[row, column / 128]
  float* ys;                   // [rows, ys_stride] power-of-two scales
  int ys_stride;
  int* err;
  int* sched;                  // [2] work-item counters of the gate/up and down launches (zeroed before each launch pair)
  unsigned long long* clk;     // [4] {SM cycles, ns} of CTA 0 summed over gate/up launches, then over down launches
};

__device__ __forceinline__ int slot_of(const GemmArgs& g, int e) { return e == g.E ? 0 : 1 + (e - g.e_own0) % g.n_stage; }
__device__ __forceinline__ int rows_of(const GemmArgs& g, int e) { return e == g.E ? g.shared_rows : g.counts[e]; }

__device__ __forceinline__ float e4m3_to_float(uint8_t c) {
  __half_raw h = __nv_cvt_fp8_to_halfraw(c, __NV_E4M3);
  return __half2float(*reinterpret_cast<__half*>(&h));
}

__device__ __forceinline__ float silu_mul(float g, float u) { return g / (1.0f + expf(-g)) * u; }

// kMode 0: gate/up + SwiGLU + requant -> hq, hs.  kMode 1: down -> y (block-scaled fp16).
// Block: 32 rows x 128 output channels, 256 threads; thread (ty, tx) owns rows ty*4..+3 and
// channels tx, tx+32, tx+64, tx+96, so one warp covers all 128 channels of its 4 rows.
template <int kMode>
__global__ void __launch_bounds__(256) gemm_simt_kernel(GemmArgs g) {
  constexpr int BR = 32, BC = 128, KS = 32;
  __shared__ float As[BR][KS + 1];
  __shared__ float Bs[kMode == 0 ? 2 : 1][BC][KS + 1];
  const int mt = g.tile_start[g.e_begin] + blockIdx.y / 4;  // 128-row tile, split in 4 sub-tiles
  if (mt >= g.tile_start[g.e_end]) return;
  const int e = g.tile_expert[mt];
  const int sub = blockIdx.y % 4;
  const int row0 = g.row_start[e] + (mt - g.tile_start[e]) * 128 + sub * BR;
  const int nrows = rows_of(g, e) - (mt - g.tile_start[e]) * 128 - sub * BR;  // valid rows from row0
  if (nrows <= 0) return;
  const int K = kMode == 0 ? g.H : g.I;
  const int N = kMode == 0 ? g.I : g.H;
  const int nb = blockIdx.x;  // 128-channel block of the output
  if (nb * BC >= N) return;
  // pool = [gate of all slots | up of all slots | down of all slots]
  const size_t IH = static_cast<size_t>(g.I) * g.H, sl = slot_of(g, e);
  const uint8_t* B0 = g.pool + ((kMode == 0 ? 0 : 2) * static_cast<size_t>(g.n_slots) + sl) * IH + static_cast<size_t>(nb) * BC * K;
  const uint8_t* B1 = g.pool + (static_cast<size_t>(g.n_slots) + sl) * IH + static_cast<size_t>(nb) * BC * K;  // up (mode 0 only)
  const int nkb = K / kBlock, nnb = N / kBlock;
  const float* s0 = (kMode == 0 ? g.gate_s : g.down_s) + (static_cast<size_t>(e) * nnb + nb) * nkb;
  const float* s1 = g.up_s + (static_cast<size_t>(e) * nnb + nb) * nkb;

  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  float acc0[4][4] = {}, acc1[4][4] = {};
  for (int kb = 0; kb < nkb; ++kb) {
    float p0[4][4] = {}, p1[4][4] = {};
    for (int ks = 0; ks < kBlock; ks += KS) {
      const int kk = kb * kBlock + ks;
      for (int i = tid; i < BR * KS; i += 256) {
        int r = i / KS, c = i % KS;
        As[r][c] = (r < nrows) ? e4m3_to_float(g.a_q[static_cast<size_t>(row0 + r) * K + kk + c]) : 0.f;
      }
      for (int i = tid; i < BC * KS; i += 256) {
        int r = i / KS, c = i % KS;
        Bs[0][r][c] = e4m3_to_float(B0[static_cast<size_t>(r) * K + kk + c]);
        if (kMode == 0) Bs[1][r][c] = e4m3_to_float(B1[static_cast<size_t>(r) * K + kk + c]);
      }
      __syncthreads();
#pragma unroll 8
      for (int c = 0; c < KS; ++c) {
        float a[4], b0[4], b1[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = As[ty * 4 + i][c];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          b0[j] = Bs[0][tx + 32 * j][c];
          if (kMode == 0) b1[j] = Bs[1][tx + 32 * j][c];
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            p0[i][j] = fmaf(a[i], b0[j], p0[i][j]);
            if (kMode == 0) p1[i][j] = fmaf(a[i], b1[j], p1[i][j]);
          }
      }
      __syncthreads();
    }
    const float w0 = s0[kb], w1 = kMode == 0 ? s1[kb] : 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = ty * 4 + i;
      const float sa = (r < nrows) ? g.a_s[static_cast<size_t>(row0 + r) * g.a_s_stride + kb] : 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        acc0[i][j] = fmaf(p0[i][j], sa * w0, acc0[i][j]);
        if (kMode == 0) acc1[i][j] = fmaf(p1[i][j], sa * w1, acc1[i][j]);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = ty * 4 + i;
    const size_t row = static_cast<size_t>(row0 + r);
    if (kMode == 0) {
      float h[4], amax = 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        h[j] = silu_mul(acc0[i][j], acc1[i][j]);
        amax = fmaxf(amax, fabsf(h[j]));
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xFFFFFFFFu, amax, off));
      const float s = (amax == 0.f) ? 1.0f : __fdiv_rn(amax, 448.0f);
      if (r < nrows) {
#pragma unroll
        for (int j = 0; j < 4; ++j)
          g.hq[row * g.I + nb * BC + tx + 32 * j] =
              static_cast<uint8_t>(__nv_cvt_float_to_fp8(__fdiv_rn(h[j], s), __NV_SATFINITE, __NV_E4M3));
        if (tx == 0) g.hs[row * g.hs_stride + nb] = s;
      }
    } else {
      // block-scaled fp16, same rule as the tensor-core kernel: amax of the row's 128 columns into [2^14, 2^15)
      float amax = 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) amax = fmaxf(amax, fabsf(acc0[i][j]));
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xFFFFFFFFu, amax, off));
      const uint32_t eb = max(__float_as_uint(amax) >> 23, 14u);
      const float mult = __uint_as_float((268u - eb) << 23);
      if (r < nrows) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const __half hv = __float2half_rn(acc0[i][j] * mult);
          g.y[row * g.H + nb * BC + tx + 32 * j] = *reinterpret_cast<const uint16_t*>(&hv);
        }
        if (tx == 0) g.ys[row * g.ys_stride + nb] = __uint_as_float((eb - 14u) << 23);
      }
    }
  }
}

}  // namespace slp
