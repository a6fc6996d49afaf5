// kernels_route.cuh — router (a1), histogram/scan/permute (a2), hidden quantisation (a3) and the
// weighted combine (a9) of the SLP MoE layer.  See DESIGN.md §6 for the per-kernel rooflines.
#pragma once
#include <cstdint>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cuda_fp16.h>

namespace slp {

constexpr int kBlock = 128;        // scale-block length
constexpr int kChunkTokens = 128;  // tokens one warp ranks in the permute kernels
constexpr int kMaxExperts = 512;

__device__ __forceinline__ float bf16_bits_to_float(uint16_t b) { return __uint_as_float(static_cast<uint32_t>(b) << 16); }

// ---------------------------------------------------------------------------------------------
// a1 (first half): router logits[t, e] = sum_h x[t, h] * W_r[e, h], fp32 FMA, fp32 accumulate.
// x is bf16 (exact in fp32).  64x64 output tile per block, 16-deep K steps, 4x4 per thread.
// ("A learned gating mechanism selects ... top-k or grouped top-k".)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) router_logits_kernel(const uint16_t* __restrict__ x, const float* __restrict__ w,
                                                            float* __restrict__ logits, int T, int H, int E) {
  constexpr int BM = 64, BN = 64, BK = 16;
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN + 4];
  const int t0 = blockIdx.x * BM, e0 = blockIdx.y * BN;
  const int tid = threadIdx.x, tx = tid % 16, ty = tid / 16;
  float acc[4][4] = {};
  const int lr = tid / 4, lc = (tid % 4) * 4;  // loader: row 0..63, 4 consecutive k
  for (int k0 = 0; k0 < H; k0 += BK) {
    {
      int t = t0 + lr;
      float v[4] = {0, 0, 0, 0};
      if (t < T) {
        uint2 raw = *reinterpret_cast<const uint2*>(x + static_cast<size_t>(t) * H + k0 + lc);
        v[0] = bf16_bits_to_float(raw.x & 0xFFFF); v[1] = bf16_bits_to_float(raw.x >> 16);
        v[2] = bf16_bits_to_float(raw.y & 0xFFFF); v[3] = bf16_bits_to_float(raw.y >> 16);
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) As[lc + i][lr] = v[i];
      int e = e0 + lr;
      float4 wv = make_float4(0, 0, 0, 0);
      if (e < E) wv = *reinterpret_cast<const float4*>(w + static_cast<size_t>(e) * H + k0 + lc);
      Bs[lc + 0][lr] = wv.x; Bs[lc + 1][lr] = wv.y; Bs[lc + 2][lr] = wv.z; Bs[lc + 3][lr] = wv.w;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int t = t0 + ty * 4 + i;
    if (t >= T) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int e = e0 + tx * 4 + j;
      if (e < E) logits[static_cast<size_t>(t) * E + e] = acc[i][j];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// a1 (second half): scores, group-limited selection and weights; one warp per token.
// Lane l holds experts l, l+32, ...  Ties go to the lower index (Q3).
//   sigmoid_bias: s = sigmoid(logit), sel = s + bias; groups scored by their two best sel;
//                 topk_group best groups kept, the rest excluded; top_k best sel among kept;
//                 w_j = s_j (/ sum) * scale.
//   softmax:      selection by logit (monotone in p); w_j = exp(l_j - max) / Z, with Z the sum
//                 over the selected (norm_topk) or over all experts.
// ---------------------------------------------------------------------------------------------
struct ArgMax {
  float v;
  int i;
};
__device__ __forceinline__ ArgMax warp_argmax(float v, int i) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    float ov = __shfl_xor_sync(0xFFFFFFFFu, v, off);
    int oi = __shfl_xor_sync(0xFFFFFFFFu, i, off);
    if (ov > v || (ov == v && oi < i)) { v = ov; i = oi; }
  }
  return {v, i};
}

template <int kPerLane>
__global__ void __launch_bounds__(256) router_topk_kernel(const float* __restrict__ logits, const float* __restrict__ bias,
                                                          int32_t* __restrict__ idx, float* __restrict__ wout, int T, int E,
                                                          int k, int G, int Gk, int scoring, int norm_topk, float scale) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= T) return;
  const float NEG = -INFINITY;
  float s[kPerLane], sel[kPerLane];
  float lmax = NEG;
#pragma unroll
  for (int r = 0; r < kPerLane; ++r) {
    int e = lane + 32 * r;
    float l = (e < E) ? logits[static_cast<size_t>(t) * E + e] : NEG;
    s[r] = l;
    lmax = fmaxf(lmax, l);
  }
  if (scoring == 0) {
#pragma unroll
    for (int r = 0; r < kPerLane; ++r) {
      int e = lane + 32 * r;
      if (e < E) {
        float sc = 1.0f / (1.0f + expf(-s[r]));
        s[r] = sc;
        sel[r] = sc + (bias ? bias[e] : 0.0f);
      } else {
        sel[r] = NEG;
      }
    }
  } else {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) lmax = fmaxf(lmax, __shfl_xor_sync(0xFFFFFFFFu, lmax, off));
    float z = 0.f;
#pragma unroll
    for (int r = 0; r < kPerLane; ++r) {
      int e = lane + 32 * r;
      sel[r] = (e < E) ? s[r] : NEG;             // select by logit
      s[r] = (e < E) ? expf(s[r] - lmax) : 0.f;  // unnormalised probability
      z += s[r];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) z += __shfl_xor_sync(0xFFFFFFFFu, z, off);
    if (!norm_topk) {
      float inv = 1.0f / z;
#pragma unroll
      for (int r = 0; r < kPerLane; ++r) s[r] *= inv;
    }
  }

  if (G > 1) {
    const int gs = E / G;
    float my_gscore = NEG;  // lane g (< G) keeps group g's score; G <= 32 checked at create
    for (int g = 0; g < G; ++g) {
      float m1 = NEG, m2 = NEG;
#pragma unroll
      for (int r = 0; r < kPerLane; ++r) {
        int e = lane + 32 * r;
        if (e < E && e / gs == g) {
          float v = sel[r];
          if (v > m1) { m2 = m1; m1 = v; } else if (v > m2) { m2 = v; }
        }
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        float o1 = __shfl_xor_sync(0xFFFFFFFFu, m1, off);
        float o2 = __shfl_xor_sync(0xFFFFFFFFu, m2, off);
        float n1 = fmaxf(m1, o1);
        float n2 = fmaxf(fminf(m1, o1), fmaxf(m2, o2));
        m1 = n1; m2 = n2;
      }
      float gsc = (gs >= 2) ? (m1 + m2) : m1;
      if (lane == g) my_gscore = gsc;
    }
    uint32_t keep = 0;
    for (int i = 0; i < Gk; ++i) {
      ArgMax a = warp_argmax(my_gscore, lane);
      keep |= 1u << a.i;
      if (lane == a.i) my_gscore = NEG;
    }
#pragma unroll
    for (int r = 0; r < kPerLane; ++r) {
      int e = lane + 32 * r;
      if (e < E && !((keep >> (e / gs)) & 1u)) sel[r] = NEG;
    }
  }

  float my_w = 0.f;
  int my_e = 0;
  float wsum = 0.f;
  for (int j = 0; j < k; ++j) {
    float bv = NEG;
    int bi = 0x7FFFFFFF;
#pragma unroll
    for (int r = 0; r < kPerLane; ++r) {
      int e = lane + 32 * r;
      if (e < E && (sel[r] > bv || (sel[r] == bv && e < bi))) { bv = sel[r]; bi = e; }
    }
    ArgMax a = warp_argmax(bv, bi);
    float sc = 0.f;
#pragma unroll
    for (int r = 0; r < kPerLane; ++r) {
      int e = lane + 32 * r;
      if (e == a.i) { sc = s[r]; sel[r] = NEG; }
    }
    sc = __shfl_sync(0xFFFFFFFFu, sc, a.i & 31);
    wsum += sc;
    if (lane == j) { my_w = sc; my_e = a.i; }
  }
  if (lane < k) {
    float wv = norm_topk ? my_w / wsum : my_w;
    idx[static_cast<size_t>(t) * k + lane] = my_e;
    wout[static_cast<size_t>(t) * k + lane] = wv * scale;
  }
}

// Same selection for the common layouts (E = 32 * kP, n_group a power of two <= 32): lane l holds the
// kP CONTIGUOUS experts l*kP .. l*kP+kP-1, so an expert group is a run of 32 / G lanes and all G
// group scores (sum of the two best sel of the group) come out of log2(32 / G) shuffle steps at once
// instead of G full-warp reductions; the kept groups follow from each group's rank among the G
// scores (ties to the lower group, as the iterative arg-max of the general kernel).  Identical
// results: same score formulas, same tie-breaks, same order of the weight sum.
template <int kP>
__global__ void __launch_bounds__(256) router_topk_fast_kernel(const float* __restrict__ logits, const float* __restrict__ bias,
                                                               int32_t* __restrict__ idx, float* __restrict__ wout, int T, int k,
                                                               int G, int Gk, int scoring, int norm_topk, float scale) {
  constexpr int E = 32 * kP;
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= T) return;
  const float NEG = -INFINITY;
  const int e0 = lane * kP;
  float s[kP], sel[kP];
  {
    const float* row = logits + static_cast<size_t>(t) * E + e0;
    if (kP % 4 == 0) {
#pragma unroll
      for (int r = 0; r < kP; r += 4) {
        const float4 v = *reinterpret_cast<const float4*>(row + r);
        s[r] = v.x; s[r + 1 < kP ? r + 1 : r] = v.y; s[r + 2 < kP ? r + 2 : r] = v.z; s[r + 3 < kP ? r + 3 : r] = v.w;
      }
    } else {
#pragma unroll
      for (int r = 0; r < kP; ++r) s[r] = row[r];
    }
  }
  if (scoring == 0) {
#pragma unroll
    for (int r = 0; r < kP; ++r) {
      const float sc = 1.0f / (1.0f + expf(-s[r]));
      s[r] = sc;
      sel[r] = sc + (bias ? bias[e0 + r] : 0.0f);
    }
  } else {
    float lmax = NEG;
#pragma unroll
    for (int r = 0; r < kP; ++r) lmax = fmaxf(lmax, s[r]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) lmax = fmaxf(lmax, __shfl_xor_sync(0xFFFFFFFFu, lmax, off));
    float z = 0.f;
#pragma unroll
    for (int r = 0; r < kP; ++r) {
      sel[r] = s[r];                 // select by logit
      s[r] = expf(s[r] - lmax);      // unnormalised probability
      z += s[r];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) z += __shfl_xor_sync(0xFFFFFFFFu, z, off);
    if (!norm_topk) {
      const float inv = 1.0f / z;
#pragma unroll
      for (int r = 0; r < kP; ++r) s[r] *= inv;
    }
  }

  if (G > 1) {
    const int lpg = 32 / G;  // lanes per group
    float m1 = NEG, m2 = NEG;
#pragma unroll
    for (int r = 0; r < kP; ++r) {
      const float v = sel[r];
      if (v > m1) { m2 = m1; m1 = v; } else if (v > m2) { m2 = v; }
    }
    for (int off = lpg >> 1; off > 0; off >>= 1) {
      const float o1 = __shfl_xor_sync(0xFFFFFFFFu, m1, off);
      const float o2 = __shfl_xor_sync(0xFFFFFFFFu, m2, off);
      const float n1 = fmaxf(m1, o1);
      const float n2 = fmaxf(fminf(m1, o1), fmaxf(m2, o2));
      m1 = n1; m2 = n2;
    }
    const float gsc = (kP * lpg >= 2) ? (m1 + m2) : m1;  // every lane of a group now holds its score
    const int g = lane / lpg;
    int rank = 0;
    for (int o = 0; o < G; ++o) {
      const float os = __shfl_sync(0xFFFFFFFFu, gsc, o * lpg);
      rank += (os > gsc || (os == gsc && o < g)) ? 1 : 0;
    }
    if (rank >= Gk) {
#pragma unroll
      for (int r = 0; r < kP; ++r) sel[r] = NEG;
    }
  }

  float my_w = 0.f;
  int my_e = 0;
  float wsum = 0.f;
  for (int j = 0; j < k; ++j) {
    float bv = NEG;
    int br = 0;
#pragma unroll
    for (int r = 0; r < kP; ++r) {  // ascending index, strict >: ties to the lower expert
      const bool better = sel[r] > bv;
      bv = better ? sel[r] : bv;
      br = better ? r : br;
    }
    // an all-excluded lane offers (-inf, its first expert); a real candidate always beats it or ties with a lower index
    const ArgMax a = warp_argmax(bv, e0 + br);
    float sc = 0.f;
#pragma unroll
    for (int r = 0; r < kP; ++r) {
      const bool hit = e0 + r == a.i;
      sc = hit ? s[r] : sc;
      sel[r] = hit ? NEG : sel[r];
    }
    sc = __shfl_sync(0xFFFFFFFFu, sc, a.i / kP);
    wsum += sc;
    if (lane == j) { my_w = sc; my_e = a.i; }
  }
  if (lane < k) {
    const float wv = norm_topk ? my_w / wsum : my_w;
    idx[static_cast<size_t>(t) * k + lane] = my_e;
    wout[static_cast<size_t>(t) * k + lane] = wv * scale;
  }
}

// ---------------------------------------------------------------------------------------------
// a2: histogram / scan / permute.  Workspace rows: [0, Tpad) hold the un-permuted tokens (the
// shared expert's rows), then each routed expert owns a 128-aligned row range holding its tokens
// in ascending token id ("sorted to form per-expert token lists").
//   pass 1: per-chunk (128 tokens, one warp) expert histograms
//   pass 2: one block: per-expert exclusive scan over chunks, counts, padded row_start,
//           tile_start and the tile -> expert table
//   pass 3: per chunk, stable ranks via match_any -> pos[t, j], row_token[row]
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) permute_hist_kernel(const int32_t* __restrict__ idx, int32_t* __restrict__ chunk_counts,
                                                           int T, int k, int E) {
  extern __shared__ int32_t sm_hist[];  // [warps][E]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int chunk = blockIdx.x * (blockDim.x >> 5) + warp;
  int32_t* h = sm_hist + warp * E;
  for (int e = lane; e < E; e += 32) h[e] = 0;
  __syncwarp();
  const int t0 = chunk * kChunkTokens;
  const int n = max(0, min(kChunkTokens, T - t0)) * k;
  const int32_t* src = idx + static_cast<size_t>(t0) * k;
  for (int i = lane; i < n; i += 32) atomicAdd(&h[src[i]], 1);
  __syncwarp();
  if (t0 < T)
    for (int e = lane; e < E; e += 32) chunk_counts[static_cast<size_t>(chunk) * E + e] = h[e];
}

// Expert sharding (the paper's SmallEP: every rank gates and sorts the full batch and keeps only
// the tokens of its own experts): experts outside [e_own0, e_own1) keep their true count in counts[] but get no
// rows and no tiles.  The shared expert covers the token range [sh_t0, sh_t1) (all tokens on one GPU, this
// rank's token shard under SmallEP, empty = no shared expert).
__global__ void __launch_bounds__(512) permute_scan_kernel(int32_t* __restrict__ chunk_counts, int32_t* __restrict__ counts,
                                                           int32_t* __restrict__ row_start, int32_t* __restrict__ tile_start,
                                                           int32_t* __restrict__ tile_expert, int32_t* __restrict__ pair_start,
                                                           int32_t* __restrict__ pair_expert, int4* __restrict__ tile_info,
                                                           int n_chunks, int T, int E, int e_own0, int e_own1, int sh_t0, int sh_t1) {
  __shared__ int32_t s_cnt[kMaxExperts + 1];   // rows that get workspace rows (0 for experts of other ranks)
  __shared__ int32_t s_tile[kMaxExperts + 2];
  __shared__ int32_t s_row[kMaxExperts + 2];
  __shared__ int32_t s_pair[kMaxExperts + 2];  // prefix of ceil(m tiles / 2): work items of the CTA-pair GEMM
  const int e = threadIdx.x;
  if (e < E) {
    int run = 0;
    for (int c0 = 0; c0 < n_chunks; c0 += 32) {  // 32 independent loads in flight, then the serial scan
      int v[32];
#pragma unroll
      for (int u = 0; u < 32; ++u) v[u] = (c0 + u < n_chunks) ? chunk_counts[static_cast<size_t>(c0 + u) * E + e] : 0;
#pragma unroll
      for (int u = 0; u < 32; ++u) {
        if (c0 + u < n_chunks) chunk_counts[static_cast<size_t>(c0 + u) * E + e] = run;
        run += v[u];
      }
    }
    s_cnt[e] = (e >= e_own0 && e < e_own1) ? run : 0;
    counts[e] = run;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const int Tpad = (T + 127) / 128 * 128;
    int row = Tpad, tile = 0, pair = 0;
    for (int i = 0; i < E; ++i) {
      row_start[i] = row;
      s_row[i] = row;
      s_tile[i] = tile;
      s_pair[i] = pair;
      int mt = (s_cnt[i] + 127) / 128;
      row += mt * 128;
      tile += mt;
      pair += (mt + 1) / 2;
    }
    const int sh_rows = max(0, sh_t1 - sh_t0), sh_tiles = (sh_rows + 127) / 128;
    row_start[E] = sh_t0;  // shared expert: the un-permuted rows of its token range
    s_row[E] = sh_t0;
    s_cnt[E] = sh_rows;
    s_tile[E] = tile;
    s_pair[E] = pair;
    tile += sh_tiles;
    pair += (sh_tiles + 1) / 2;
    s_tile[E + 1] = tile;
    s_pair[E + 1] = pair;
    row_start[E + 1] = row;  // total rows in use
  }
  __syncthreads();
  for (int i = threadIdx.x; i < E + 2; i += blockDim.x) { tile_start[i] = s_tile[i]; pair_start[i] = s_pair[i]; }
  for (int i = threadIdx.x; i <= E; i += blockDim.x) {
    for (int m = s_tile[i]; m < s_tile[i + 1]; ++m) {
      tile_expert[m] = i;
      const int m_in_e = m - s_tile[i];  // one record per 128-row tile: {expert, first workspace row, valid rows, tile index in expert}
      tile_info[m] = make_int4(i, s_row[i] + m_in_e * 128, min(128, s_cnt[i] - m_in_e * 128), m_in_e);
    }
    for (int m = s_pair[i]; m < s_pair[i + 1]; ++m) pair_expert[m] = i;
  }
}

__global__ void __launch_bounds__(128) permute_place_kernel(const int32_t* __restrict__ idx, const int32_t* __restrict__ chunk_off,
                                                            const int32_t* __restrict__ row_start, int32_t* __restrict__ pos,
                                                            int32_t* __restrict__ row_token, int T, int k, int E, int e_own0, int e_own1) {
  extern __shared__ int32_t sm_run[];  // [warps][E] next free row of each expert for this chunk
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int chunk = blockIdx.x * (blockDim.x >> 5) + warp;
  const int t0 = chunk * kChunkTokens;
  if (t0 >= T) return;
  int32_t* run = sm_run + warp * E;
  for (int e = lane; e < E; e += 32) run[e] = row_start[e] + chunk_off[static_cast<size_t>(chunk) * E + e];
  __syncwarp();
  const int n = min(kChunkTokens, T - t0) * k;
  const int32_t* src = idx + static_cast<size_t>(t0) * k;
  for (int base = 0; base < n; base += 32) {
    const int i = base + lane;
    const bool valid = i < n;
    const int e = valid ? src[i] : -1 - lane;  // entries are token-major: ascending lane = ascending token
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, e);
    const int rank = __popc(peers & ((1u << lane) - 1));
    const bool own = valid && e >= e_own0 && e < e_own1;  // experts of other ranks get no row: pos = -1
    int dst = -1;
    if (own) dst = run[e] + rank;
    __syncwarp();
    if (own && rank == 0) run[e] += __popc(peers);
    __syncwarp();
    if (valid) {
      const int t = t0 + i / k;
      pos[static_cast<size_t>(t0) * k + i] = dst;
      if (own) row_token[dst] = t;
    }
  }
  for (int i = lane; i < min(kChunkTokens, T - t0); i += 32) row_token[t0 + i] = t0 + i;  // shared rows
}

// ---------------------------------------------------------------------------------------------
// a3: hidden quantisation, fused with the scatter into expert order.  Per token, per 128
// channels: amax -> s = amax / 448 -> e4m3(x / s) (fp32 IEEE division, RNE, saturating), written
// to the token's own row (shared-expert region) and to its k expert rows.
// ("activations are quantized to FP8"; Q10-Q12.)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t quant4_e4m3(float a, float b, float c, float d, float s) {
  __nv_fp8x2_storage_t lo = __nv_cvt_float2_to_fp8x2(make_float2(__fdiv_rn(a, s), __fdiv_rn(b, s)), __NV_SATFINITE, __NV_E4M3);
  __nv_fp8x2_storage_t hi = __nv_cvt_float2_to_fp8x2(make_float2(__fdiv_rn(c, s), __fdiv_rn(d, s)), __NV_SATFINITE, __NV_E4M3);
  return static_cast<uint32_t>(lo) | (static_cast<uint32_t>(hi) << 16);
}

__global__ void __launch_bounds__(256) quant_scatter_kernel(const uint16_t* __restrict__ x, const int32_t* __restrict__ pos,
                                                            uint8_t* __restrict__ xq, float* __restrict__ xs, int T, int H, int k,
                                                            int xs_stride) {
  // One block per token; a half-warp owns a 128-channel block (8 channels = one 16-byte load per lane),
  // so a warp quantises two blocks per step: half the instructions per byte of a lane-per-4-channels
  // layout (the kernel is issue-bound on the IEEE divisions, not on HBM).
  const int t = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
  const int sub = lane >> 4, l16 = lane & 15;
  __shared__ int32_t dst[33];
  if (threadIdx.x < k) dst[threadIdx.x + 1] = pos[static_cast<size_t>(t) * k + threadIdx.x];
  if (threadIdx.x == 0) dst[0] = t;
  __syncthreads();
  const int nkb = H / kBlock;
  for (int kb0 = warp * 2; kb0 < nkb; kb0 += nwarps * 2) {
    const int kb = kb0 + sub;
    const bool on = kb < nkb;  // odd number of blocks: the upper half-warp idles in the last step
    uint4 raw = make_uint4(0u, 0u, 0u, 0u);
    if (on) raw = *reinterpret_cast<const uint4*>(x + static_cast<size_t>(t) * H + kb * kBlock + l16 * 8);
    float v[8];
    v[0] = bf16_bits_to_float(raw.x & 0xFFFF); v[1] = bf16_bits_to_float(raw.x >> 16);
    v[2] = bf16_bits_to_float(raw.y & 0xFFFF); v[3] = bf16_bits_to_float(raw.y >> 16);
    v[4] = bf16_bits_to_float(raw.z & 0xFFFF); v[5] = bf16_bits_to_float(raw.z >> 16);
    v[6] = bf16_bits_to_float(raw.w & 0xFFFF); v[7] = bf16_bits_to_float(raw.w >> 16);
    float amax = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) amax = fmaxf(amax, fabsf(v[i]));
#pragma unroll
    for (int off = 8; off > 0; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xFFFFFFFFu, amax, off));  // within the half-warp
    const float s = (amax == 0.f) ? 1.0f : __fdiv_rn(amax, 448.0f);
    const uint2 q = make_uint2(quant4_e4m3(v[0], v[1], v[2], v[3], s), quant4_e4m3(v[4], v[5], v[6], v[7], s));
    if (on) {
      for (int j = 0; j <= k; ++j) {
        if (dst[j] < 0) continue;  // expert owned by another rank (SmallEP): no row here
        const size_t row = dst[j];
        *reinterpret_cast<uint2*>(xq + row * H + kb * kBlock + l16 * 8) = q;
        if (l16 == 0) xs[row * xs_stride + kb] = s;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// a9: weighted combine.  out[t] = sum_j w[t,j] * Y[pos[t,j]] (fixed j order, fp32 FMA) + Y[t]
// (shared expert row, weight 1).  Y rows are block-scaled fp16 (y = y16 * ys[row, column / 128], ys a power
// of two), the sum is fp32 and rounded once to bf16.  Gather-based, no atomics.
// (PAPER.md:92 step 5 "A final weighted sum"; "router-weighted accumulation in F32".)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void fma_f16x8(float (&acc)[8], float s, const uint4& v) {
  const uint32_t u[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&u[i]));
    acc[2 * i] = fmaf(s, f.x, acc[2 * i]);
    acc[2 * i + 1] = fmaf(s, f.y, acc[2 * i + 1]);
  }
}

// kPartial (SmallEP): slots whose expert lives on another rank have pos < 0 and are skipped, the shared
// expert is added only for tokens in [sh_t0, sh_t1), and the fp32 sum is written unrounded: the ranks'
// partial sums are reduced first ("partial weighted sum ... exchange and local reduction")
// and rounded to bf16 once, by partial_to_bf16_kernel.
template <bool kPartial>
__global__ void __launch_bounds__(256) combine_kernel(const uint16_t* __restrict__ y, const float* __restrict__ ys, const int32_t* __restrict__ pos,
                                                      const float* __restrict__ w, void* __restrict__ out, int T, int H,
                                                      int k, int sh_t0, int sh_t1, int ys_stride) {
  const int t = blockIdx.x;
  __shared__ int32_t s_row[32];
  __shared__ float s_w[32];
  if (threadIdx.x < k) {
    s_row[threadIdx.x] = pos[static_cast<size_t>(t) * k + threadIdx.x];
    s_w[threadIdx.x] = w[static_cast<size_t>(t) * k + threadIdx.x];
  }
  __syncthreads();
  const bool has_shared = t >= sh_t0 && t < sh_t1;
  for (int c = threadIdx.x * 8; c < H; c += blockDim.x * 8) {  // 8 channels = one 16-byte load per row
    float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (int j = 0; j < k; ++j) {
      if (kPartial && s_row[j] < 0) continue;
      const size_t row = s_row[j];
      const uint4 v = *reinterpret_cast<const uint4*>(y + row * H + c);
      fma_f16x8(acc, s_w[j] * ys[row * ys_stride + (c >> 7)], v);  // power-of-two block scale: the product is exact
    }
    if (has_shared) {
      const uint4 v = *reinterpret_cast<const uint4*>(y + static_cast<size_t>(t) * H + c);
      fma_f16x8(acc, ys[static_cast<size_t>(t) * ys_stride + (c >> 7)], v);
    }
    if (kPartial) {
      float4* dst = reinterpret_cast<float4*>(static_cast<float*>(out) + static_cast<size_t>(t) * H + c);
      dst[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
      dst[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
    } else {
      uint4 o;
      __nv_bfloat162 p0 = __floats2bfloat162_rn(acc[0], acc[1]), p1 = __floats2bfloat162_rn(acc[2], acc[3]);
      __nv_bfloat162 p2 = __floats2bfloat162_rn(acc[4], acc[5]), p3 = __floats2bfloat162_rn(acc[6], acc[7]);
      o.x = *reinterpret_cast<uint32_t*>(&p0); o.y = *reinterpret_cast<uint32_t*>(&p1);
      o.z = *reinterpret_cast<uint32_t*>(&p2); o.w = *reinterpret_cast<uint32_t*>(&p3);
      *reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(out) + static_cast<size_t>(t) * H + c) = o;
    }
  }
}

// The one bf16 rounding of the SmallEP path: reduced fp32 partial sums -> bf16 (n a multiple of 4).
__global__ void __launch_bounds__(256) partial_to_bf16_kernel(const float* __restrict__ sum, __nv_bfloat16* __restrict__ out, size_t n4) {
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < n4; i += static_cast<size_t>(gridDim.x) * blockDim.x) {
    const float4 v = reinterpret_cast<const float4*>(sum)[i];
    __nv_bfloat162 lo = __floats2bfloat162_rn(v.x, v.y), hi = __floats2bfloat162_rn(v.z, v.w);
    reinterpret_cast<uint2*>(out)[i] = make_uint2(*reinterpret_cast<uint32_t*>(&lo), *reinterpret_cast<uint32_t*>(&hi));
  }
}

}  // namespace slp
