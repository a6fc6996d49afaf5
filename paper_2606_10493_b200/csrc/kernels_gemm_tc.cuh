// kernels_gemm_tc.cuh — grouped FP8 GEMM on the 5th-gen tensor cores (a5, a6, a7, a8).
//
// One persistent CTA per SM works through the (128-row tile, N tile) work items of the experts of the
// launch (one 16-byte record per tile, written by permute_scan_kernel); an otherwise idle warp takes the
// items from a global counter, so all CTAs stay within ~gridDim consecutive items and share operands
// through L2 (SLP_TRIAGE gemm=static: static round-robin instead).  Per
// 128-deep K block the tensor core writes a fresh 128 x 256 fp32 partial into one of two TMEM
// buffers; the promotion warps pull it out with tcgen05.ld and add it into fp32 register accumulators
// with one FMA per element (issued as FFMA2 pairs), scaled by  xs[row, kb] * ws[n-block, kb]
// ("FP8 GEMM with FP32 accumulation"; "accumulate all partial dot-products
// first and apply the scale once per block").
//
//   warp 8      TMA producer (one elected thread): A tile (128 rows x 128 B) + 64-row B boxes per K
//               block into a 128B-swizzled smem ring (mbarrier full / empty)
//   warp 9      MMA issuer (one elected thread): per K block 4 x tcgen05.mma.kind::f8f6f4 (M128 N256
//               K32) into TMEM buffer kb mod 2; tcgen05.commit publishes the buffer and frees the stage
//   warp 10     work scheduler (one elected thread): atomicAdd on the launch's counter -> 4-deep smem ring
//               read by the producer, the MMA issuer and the promotion warps
//   warp 11     idle (warps 8-11 donate most of their registers to the promotion warps, setmaxnreg)
//   warps 0-7   promotion + epilogue: warp w owns TMEM lanes 32 * (w % 4).. (rows) and the 128 columns
//               of half w / 4; 128 fp32 accumulators per thread; the TMEM buffer is handed back as
//               soon as the last tcgen05.ld has landed, before the last FMAs
//
// kPair (SLP_TRIAGE gemm=pair): a cluster of two CTAs issues ONE cta_group::2 MMA with M = 256 (two
//   128-row tiles of the same expert) x N = 256; each CTA stages its own A tile and half of the B tile
//   (TMA loads of both CTAs complete on the leader's mbarrier, commits are multicast to both CTAs, the
//   peer's promotion warps release TMEM on the leader's barrier).  It moves a third less operand data
//   per MAC from L2 and through the shared-memory port; see DESIGN.md §6.1 for where each variant stands.
//
// All barrier / stage addresses are 32-bit shared-window addresses computed once (ptx::launder_u32):
// re-deriving them from generic pointers cost ~100 of the ~285 instructions per warp per K block.
//
// kMode 0 (gate/up): B smem rows = [gate n0..+63 | up n0..+63 | gate n0+64..+127 | up n0+64..+127],
//   so each half holds the gate and up columns of the same 64 intermediate channels; epilogue
//   h = silu(g) * u, row amax over the 128 channels (two halves, exchanged through smem),
//   s = amax / 448, e4m3(h / s) -> hq, hs  ("SiLU(.) (.)"; Q14).
// kMode 1 (down):   B = down rows n0..n0+255; epilogue: the Y tile is stored as block-scaled fp16 (one
//   power-of-two scale per row per 128 columns), staged whole in shared memory and leaves through TMA
//   stores while the next tile's K loop runs.
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
constexpr int kBoxRows = 64;  // rows per B TMA box
constexpr int kEpiWarps = 8;
constexpr int kThreads = (kEpiWarps + 4) * 32;  // three warpgroups: 2 x promotion, 1 x {producer, MMA, 2 idle}
constexpr int kTmemCols = 512;
constexpr int kMaxStages = 6;
constexpr int kSchedDepth = 4;  // work items the scheduler warp may run ahead of the roles

// kPair = false: one CTA per tile, A tile (16 KB) + whole B tile (32 KB) per stage, 4 stages.
// kPair = true:  a cluster of two CTAs issues one cta_group::2 MMA with M = 256 (two 128-row tiles
//                of the same expert) x N = 256; each CTA stages its own A tile and HALF of the B tile
//                (16 KB + 16 KB per stage, 6 stages), which cuts the L2 -> SM operand traffic per MAC
//                by a third (the 1-CTA kernel is L2-bandwidth bound, profiles/r1_gemm_baseline.md).
template <int kMode, bool kPair> struct Cfg {
  // The down kernel trades one pipeline stage for a staging area that holds its whole fp16 Y tile
  // (64 KB): its tiles are only 16 K blocks long, so the epilogue must not wait on TMA-store read-out.
  static constexpr int kStages = kPair ? (kMode == 1 ? 5 : 6) : (kMode == 1 ? 3 : 4);
  static constexpr int kABytes = BM * BK;
  static constexpr int kBBytes = (kPair ? BN / 2 : BN) * BK;
  static constexpr int kStageBytes = kABytes + kBBytes;
  static constexpr int kScratchBytes = kMode == 1 ? kEpiWarps * 8192 : 32768;  // mode 1: the whole fp16 Y tile (two 4 KB boxes per warp); mode 0: amax exchange only
  static constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 256 /*barriers*/ + kScratchBytes;
  static_assert(kSmemBytes <= 232448, "shared memory budget");
};

// Barrier block behind the stage ring; the kernels address it through 32-bit shared addresses.
struct Shared {
  uint64_t full[kMaxStages];   // TMA -> MMA: stage landed (pair: lives in the leader CTA, fed by both CTAs' loads)
  uint64_t empty[kMaxStages];  // MMA -> TMA: stage consumed (pair: multicast commit to both CTAs)
  uint64_t tmem_full[2];       // MMA -> promotion: K block partial complete in TMEM buffer b
  uint64_t tmem_empty[2];      // promotion -> MMA: buffer b read out (pair: 2 x kEpiWarps arrivals at the leader)
  uint64_t sched_full[kSchedDepth];   // scheduler -> roles: work item published
  uint64_t sched_empty[kSchedDepth];  // roles -> scheduler: slot read by producer, MMA issuer and the promotion warps
  int32_t sched_w[kSchedDepth];       // work item of each slot (-1 = no more work)
  uint32_t tmem_base;
  int dead;
};
static_assert(sizeof(Shared) <= 256, "barrier block");
constexpr uint32_t kOffFull = 0, kOffEmpty = 8 * kMaxStages, kOffTmemFull = 16 * kMaxStages, kOffTmemEmpty = 16 * kMaxStages + 16;
constexpr uint32_t kOffSchedFull = kOffTmemEmpty + 16, kOffSchedEmpty = kOffSchedFull + 8 * kSchedDepth;

// silu(g) * u with the fast exponential and reciprocal (rel. error ~1e-6, three decades below the
// e4m3 step that follows).
__device__ __forceinline__ float silu_mul_fast(float g, float u) {
  float t, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(t) : "f"(g * -1.4426950408889634f));  // e^-g; overflow -> +inf -> r = 0
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + t));
  return g * r * u;
}

// p ? a : b as one SELP (keeps the scale bookkeeping of the K loop free of branches and copies).
__device__ __forceinline__ float sel_f32(bool p, float a, float b) {
  float r;
  asm("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %3, 0;\n\tselp.f32 %0, %1, %2, q;\n\t}" : "=f"(r) : "f"(a), "f"(b), "r"(static_cast<int>(p)));
  return r;
}

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

template <int kMode, bool kPair, bool kDyn = false>
__global__ void __launch_bounds__(kThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b,
               const __grid_constant__ CUtensorMap tm_y, GemmArgs g) {
  using C = Cfg<kMode, kPair>;
  constexpr int kStages = C::kStages, kABytes = C::kABytes, kStageBytes = C::kStageBytes, kScratchBytes = C::kScratchBytes;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* scratch = smem + kStages * kStageBytes;  // 1024-aligned: per-warp staging for the Y TMA stores / amax exchange
  Shared* sh = reinterpret_cast<Shared*>(scratch + kScratchBytes);
  const uint32_t smem_a = ptx::launder_u32(ptx::smem_u32(smem));               // stage ring base (shared window address)
  const uint32_t bar_a = ptx::launder_u32(smem_a + kStages * kStageBytes + kScratchBytes);  // barrier block base
  const uint32_t rank = kPair ? ptx::cluster_ctarank() : 0u;                   // CTA of the pair; 0 = leader (issues the MMAs)
  const uint32_t lead_bar = kPair ? ptx::launder_u32(ptx::mapa(bar_a, 0)) : bar_a;  // leader's barrier block (cluster address)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  long long clk0 = 0;
  unsigned long long ns0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {  // average SM clock of this launch (evidence for the power-capped regime)
    clk0 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns0));
  }
  const int K = kMode == 0 ? g.H : g.I;
  const int N = kMode == 0 ? g.I : g.H;
  const int num_kb = K / BK;
  const int n_tiles = kMode == 0 ? N / 128 : (N + BN - 1) / BN;
  // work items: (128-row tile | pair of tiles, N tile) over the experts of this launch
  const int it_begin = kPair ? g.pair_start[g.e_begin] : g.tile_start[g.e_begin];
  const int it_end = kPair ? g.pair_start[g.e_end] : g.tile_start[g.e_end];
  const int total = (it_end - it_begin) * n_tiles;
  const int w_first = kPair ? static_cast<int>(blockIdx.x >> 1) : static_cast<int>(blockIdx.x);
  const int w_step = kPair ? static_cast<int>(gridDim.x >> 1) : static_cast<int>(gridDim.x);

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&sh->full[i], 1); ptx::mbar_init(&sh->empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&sh->tmem_full[i], 1); ptx::mbar_init(&sh->tmem_empty[i], kPair ? 2 * kEpiWarps : kEpiWarps); }
    for (int i = 0; i < kSchedDepth; ++i) { ptx::mbar_init(&sh->sched_full[i], 1); ptx::mbar_init(&sh->sched_empty[i], 2 + kEpiWarps); }
    sh->dead = 0;
    ptx::fence_mbar_init();
  }
  if (warp == kEpiWarps + 1) {
    if (kPair) ptx::tmem_alloc_2sm<kTmemCols>(&sh->tmem_base);
    else ptx::tmem_alloc<kTmemCols>(&sh->tmem_base);
  }
  if (warp == kEpiWarps && lane == 0) { ptx::prefetch_tmap(&tm_a); ptx::prefetch_tmap(&tm_b); }
  ptx::tc_fence_before();
  __syncthreads();
  if (kPair) ptx::cluster_sync();  // the peer's barriers are initialised before anything remote touches them
  ptx::tc_fence_after();
  const uint32_t tmem_base = sh->tmem_base;
  volatile int* dead = &sh->dead;

  // Work item w -> (expert, this CTA's 128-row tile inside the expert, N tile): n fastest, so the CTAs
  // running together cover a few m tiles of one expert against all of its N tiles and share both
  // operands through L2.  One 16-byte record per tile (written by permute_scan_kernel) replaces a
  // chain of dependent loads.  Pair kernel: the second CTA of the last pair of an expert with an odd
  // number of tiles gets nrows = 0 (it re-reads the previous tile and stores nothing).
  struct Tile { int e, row0, nrows, nt; };
  auto fetch = [&](int w) {
    Tile t;
    const int item = it_begin + w / n_tiles;
    t.nt = w % n_tiles;
    if (kPair) {
      t.e = g.pair_expert[item];
      const int mt_e = g.tile_start[t.e + 1] - g.tile_start[t.e];
      int m_in_e = 2 * (item - g.pair_start[t.e]) + static_cast<int>(rank);
      const bool valid = m_in_e < mt_e;
      if (!valid) m_in_e = mt_e - 1;
      t.row0 = g.row_start[t.e] + m_in_e * BM;
      t.nrows = valid ? min(BM, rows_of(g, t.e) - m_in_e * BM) : 0;
    } else {
      const int4 ti = g.tile_info[item];
      t.e = ti.x; t.row0 = ti.y; t.nrows = ti.z;
    }
    return t;
  };

  // Next work item of this CTA after `w` (its i-th), or -1.  Static order: w + gridDim.  kDyn (one-CTA
  // kernel, the default; SLP_TRIAGE gemm=static selects the static order): items come from a global counter through a small shared-memory ring fed by an idle warp, so
  // all CTAs stay inside a window of ~gridDim consecutive items and the B tiles they share stay in L2
  // (profiles/r1_sched_ab.md).  Which CTA computes a tile does not change its result.
  auto next_item = [&](int w, int i, bool whole_warp) -> int {
    if constexpr (kPair || !kDyn) {
      w += w_step;
    } else {
      const uint32_t slot = static_cast<uint32_t>(i) % kSchedDepth;
      ptx::mbar_wait_a(bar_a + kOffSchedFull + 8 * slot, (static_cast<uint32_t>(i) / kSchedDepth) & 1, dead, g.err, 5);
      w = sh->sched_w[slot];  // plain load from a warp-uniform address (the wait above is a compiler barrier)
      if (whole_warp) {
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_a(bar_a + kOffSchedEmpty + 8 * slot);
      } else {
        ptx::mbar_arrive_a(bar_a + kOffSchedEmpty + 8 * slot);
      }
    }
    return w < total ? w : -1;
  };

  // Registers: 168 per thread at launch (384 threads); the producer / MMA warpgroup gives most of
  // its share to the two promotion warpgroups, which hold 128 accumulators + two loads in flight.
  if (warp >= kEpiWarps) {
   ptx::setmaxnreg_dec<40>();
   if (warp == kEpiWarps) {
    // ===================== TMA producer (one elected thread) =====================
    if (ptx::elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      Tile nx{0, 0, 0, 0};
      if (w_first < total) nx = fetch(w_first);  // idle CTAs (and launches without any tile) read no record
      int w = w_first < total ? w_first : -1;
      for (int i = 0; w >= 0; ++i) {
        const Tile cur = nx;
        w = next_item(w, i, false);
        if (w >= 0) nx = fetch(w);  // next tile's record is in flight during this tile's loads
        const int e = cur.e, nt = cur.nt, row0 = cur.row0;
        const int slot = slot_of(g, e);
        constexpr int kBoxes = kPair ? 2 : 4;
        int brow[kBoxes];
        if (kMode == 0) {
          // pool = [gate of all slots | up of all slots | down of all slots], viewed as [3 * slots * I, H]
          const int gate0 = slot * g.I + nt * 128, up0 = (g.n_slots + slot) * g.I + nt * 128;
          if (kPair) { brow[0] = gate0 + 64 * rank; brow[1] = up0 + 64 * rank; }
          else { brow[0] = gate0; brow[1] = up0; brow[2 % kBoxes] = gate0 + 64; brow[3 % kBoxes] = up0 + 64; }
        } else {
          const int down0 = (2 * g.n_slots + slot) * g.H + nt * BN;  // same pool viewed as [3 * slots * H, I]
          if (kPair) { brow[0] = down0 + 128 * rank; brow[1] = brow[0] + 64; }
          else { brow[0] = down0; brow[1] = down0 + 64; brow[2 % kBoxes] = down0 + 128; brow[3 % kBoxes] = down0 + 192; }
        }
        for (int kb = 0; kb < num_kb; ++kb) {
          ptx::mbar_wait_a(bar_a + kOffEmpty + 8 * stage, phase ^ 1, dead, g.err, 1);
          const uint32_t sa = smem_a + stage * kStageBytes, sb = sa + kABytes;
          if (kPair) {
            const uint32_t fb = lead_bar + kOffFull + 8 * stage;  // both CTAs' bytes complete on the leader's barrier
            if (rank == 0) ptx::mbar_arrive_expect_tx_a(bar_a + kOffFull + 8 * stage, 2 * kStageBytes);
            ptx::tma_load_2d_2sm(sa, &tm_a, fb, kb * BK, row0);
#pragma unroll
            for (int b = 0; b < kBoxes; ++b) ptx::tma_load_2d_2sm(sb + b * kBoxRows * BK, &tm_b, fb, kb * BK, brow[b]);
          } else {
            const uint32_t fb = bar_a + kOffFull + 8 * stage;
            ptx::mbar_arrive_expect_tx_a(fb, kStageBytes);
            ptx::tma_load_2d_a(sa, &tm_a, fb, kb * BK, row0);
#pragma unroll
            for (int b = 0; b < kBoxes; ++b) ptx::tma_load_2d_a(sb + b * kBoxRows * BK, &tm_b, fb, kb * BK, brow[b]);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
   } else if (warp == kEpiWarps + 2) {
    // ===================== work scheduler (kDyn; one elected thread) =====================
    if (!kPair && kDyn && ptx::elect_one()) {
      for (int i = 0;; ++i) {  // slot i holds the item that FOLLOWS this CTA's i-th item (the first is blockIdx)
        const uint32_t slot = static_cast<uint32_t>(i) % kSchedDepth;
        ptx::mbar_wait_a(bar_a + kOffSchedEmpty + 8 * slot, ((static_cast<uint32_t>(i) / kSchedDepth) & 1) ^ 1, dead, g.err, 6);
        const int w = static_cast<int>(gridDim.x) + atomicAdd(g.sched + kMode, 1);
        sh->sched_w[slot] = w;
        ptx::mbar_arrive_a(bar_a + kOffSchedFull + 8 * slot);  // release: the store above is visible to the waiters
        if (w >= total) break;
      }
    }
   } else if (warp == kEpiWarps + 1) {
    // ===================== MMA issuer (one elected thread; pair: leader CTA only) =====================
    if (rank == 0 && ptx::elect_one()) {
      constexpr uint32_t idesc = ptx::umma_idesc_e4m3_f32(kPair ? 2 * BM : BM, BN);
      const uint64_t adesc0 = ptx::umma_desc_k128_a(smem_a), bdesc0 = ptx::umma_desc_k128_a(smem_a + kABytes);
      int stage = 0;
      uint32_t phase = 0;
      uint32_t it = 0;  // running K-block counter: TMEM buffer = it & 1
      int w = w_first < total ? w_first : -1;
      for (int i = 0; w >= 0; w = next_item(w, i, false), ++i) {
        for (int kb = 0; kb < num_kb; ++kb, ++it) {
          const uint32_t buf = it & 1, tph = ((it >> 1) & 1) ^ 1;
          ptx::mbar_wait_a(bar_a + kOffFull + 8 * stage, phase, dead, g.err, 3);    // operands landed (usually long ago)
          ptx::mbar_wait_a(bar_a + kOffTmemEmpty + 8 * buf, tph, dead, g.err, 2);   // the critical hand-off: issue right after it
          ptx::tc_fence_after();
          const uint64_t so = static_cast<uint64_t>((stage * kStageBytes) >> 4);
          const uint32_t d = tmem_base + buf * BN;
#pragma unroll
          for (int k4 = 0; k4 < BK / 32; ++k4) {  // UMMA_K = 32 for 8-bit operands: +32 B per step
            if (kPair) ptx::umma_f8_2sm(d, adesc0 + so + 2 * k4, bdesc0 + so + 2 * k4, idesc, k4 > 0);
            else ptx::umma_f8(d, adesc0 + so + 2 * k4, bdesc0 + so + 2 * k4, idesc, k4 > 0);
          }
          if (kPair) {
            ptx::umma_commit_2sm_mc(bar_a + kOffTmemFull + 8 * buf, 3);  // both CTAs' halves of the partial are complete
            ptx::umma_commit_2sm_mc(bar_a + kOffEmpty + 8 * stage, 3);   // both CTAs' stages reusable once these MMAs retire
          } else {
            ptx::umma_commit_a(bar_a + kOffTmemFull + 8 * buf);
            ptx::umma_commit_a(bar_a + kOffEmpty + 8 * stage);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
   }
  } else {
    // ===================== promotion + epilogue =====================
    ptx::setmaxnreg_inc<232>();
    const int q = warp & 3, half = warp >> 2;
    const int r_in_tile = q * 32 + lane;
    const uint32_t tm_lane = ptx::launder_u32(tmem_base + (static_cast<uint32_t>(q * 32) << 16) + half * HN);
    uint32_t it = 0;
    int tile_parity = 0;
    const uint32_t te_a = lead_bar + kOffTmemEmpty;  // pair: the leader's barrier (cluster address)
    // Per-tile scale pointers; the first loads of a tile are issued before the previous tile's epilogue.
    const float *as_ptr = nullptr, *ws0 = nullptr, *ws1 = nullptr;
    bool row_ok = false;
    float4 xs_nxt = make_float4(0.f, 0.f, 0.f, 0.f);
    float w0_nxt = 0.f, w1_nxt = 0.f;
    auto open_tile = [&](const Tile& t) {
      row_ok = r_in_tile < t.nrows;
      as_ptr = g.a_s + static_cast<size_t>(t.row0 + r_in_tile) * g.a_s_stride;  // padded to a multiple of 4 floats, 16-byte aligned
      // weight-scale rows of this thread's columns: chunks 0-3 use ws0, chunks 4-7 use ws1
      if (kMode == 0) {
        const size_t o = (static_cast<size_t>(t.e) * (g.I / 128) + t.nt) * num_kb;
        ws0 = g.gate_s + o;
        ws1 = g.up_s + o;
      } else {
        const int nb = min(t.nt * 2 + half, g.H / 128 - 1);
        ws0 = g.down_s + (static_cast<size_t>(t.e) * (g.H / 128) + nb) * num_kb;
        ws1 = ws0;
      }
      // Scales are fetched far ahead of use: the row's activation scales four K blocks at a time
      // (one 16-byte load), the weight scales 32 K blocks at a time, one per lane, broadcast by shuffle.
      xs_nxt = row_ok ? *reinterpret_cast<const float4*>(as_ptr) : make_float4(0.f, 0.f, 0.f, 0.f);
      w0_nxt = lane < num_kb ? ws0[lane] : 0.f;
      w1_nxt = (kMode == 0 && lane < num_kb) ? ws1[lane] : 0.f;
    };
    Tile nx{0, 0, 0, 0};
    if (w_first < total) { nx = fetch(w_first); open_tile(nx); }
    int w = w_first < total ? w_first : -1;
#ifdef SLP_PROF
    long long pk = 0, pe = 0, pf = 0, pn = 0, pq = 0;
#endif
    for (int i = 0; w >= 0; ++i, tile_parity ^= 1) {
#ifdef SLP_PROF
      const long long p0 = clock64();
      long long p1 = p0;
#endif
      const Tile cur = nx;
      w = next_item(w, i, true);
      const bool has_next = w >= 0;
      if (has_next) nx = fetch(w);  // record in flight during the K loop
#ifdef SLP_PROF
      const long long pa = clock64();
#endif
      const int nt = cur.nt, row0 = cur.row0, nrows = cur.nrows;
      const size_t row = static_cast<size_t>(row0 + r_in_tile);
      const bool row_ok_cur = row_ok;
      uint64_t acc2[64];  // 128 fp32 accumulators as FFMA2 pairs
#pragma unroll
      for (int i = 0; i < 64; ++i) acc2[i] = 0ull;

      float w0_cur = 0.f, w1_cur = 0.f;
      float4 xs_cur = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
      for (int kb = 0; kb < num_kb; ++kb) {
        {
          // Branch-free scale bookkeeping (selp): a branchy version cost ~40 MOV / BRA per K block in
          // an issue-bound loop.  Every 4th K block the row's next four activation scales (one 16-byte
          // load issued a group ahead) become current; every 32nd the lane-held weight scales rotate.
          const int j = kb & 3;
          const bool g4 = j == 0, g32 = (kb & 31) == 0;
          xs_cur.x = sel_f32(g4, xs_nxt.x, xs_cur.x);
          xs_cur.y = sel_f32(g4, xs_nxt.y, xs_cur.y);
          xs_cur.z = sel_f32(g4, xs_nxt.z, xs_cur.z);
          xs_cur.w = sel_f32(g4, xs_nxt.w, xs_cur.w);
          w0_cur = sel_f32(g32, w0_nxt, w0_cur);
          w1_cur = sel_f32(g32, w1_nxt, w1_cur);
          if (g4) {
            if (kb + 4 < num_kb && row_ok) xs_nxt = *reinterpret_cast<const float4*>(as_ptr + kb + 4);
            if (g32) {
              const int kn = kb + 32 + lane;
              w0_nxt = kn < num_kb ? ws0[kn] : 0.f;
              w1_nxt = (kMode == 0 && kn < num_kb) ? ws1[kn] : 0.f;
            }
          }
          const float sa = sel_f32((j & 2) != 0, sel_f32((j & 1) != 0, xs_cur.w, xs_cur.z), sel_f32((j & 1) != 0, xs_cur.y, xs_cur.x));
          const float sc0 = sa * __shfl_sync(0xFFFFFFFFu, w0_cur, kb & 31);
          const float sc1 = kMode == 0 ? sa * __shfl_sync(0xFFFFFFFFu, w1_cur, kb & 31) : sc0;
          const uint64_t s20 = ptx::pack2(sc0, sc0), s21 = ptx::pack2(sc1, sc1);
          const uint32_t buf = it & 1;
          ptx::mbar_wait_a(bar_a + kOffTmemFull + 8 * buf, (it >> 1) & 1, dead, g.err, 4);
          ptx::tc_fence_after();
#ifdef SLP_PROF
          if (kb == 0) p1 = clock64();
#endif
          const uint32_t tb = tm_lane + buf * BN;
          {
            // 8 chunks of 16 columns through four register sets: chunks 0-3 are loaded up front, chunk
            // c + 4 is requested as soon as the FMAs of chunk c have consumed its set, so every
            // tcgen05.ld of the K block has landed after half of the FMAs and the TMEM buffer goes back
            // to the MMA issuer there.  The K loop is bound by the hand-off round trip, not by throughput:
            // time per K block = (MMA 512 + ~500 cycles of commit / wake-up / issue latency + drain) / 2
            // with two TMEM buffers, drain = buffer published -> buffer released.
            uint32_t v[4][16];
  #pragma unroll
            for (int c = 0; c < 4; ++c) ptx::tmem_ld16(tb + c * 16, v[c]);
            ptx::tmem_ld_wait16(v[0]);
            ptx::keep16(v[1]); ptx::keep16(v[2]); ptx::keep16(v[3]);
  #pragma unroll
            for (int c = 0; c < 4; ++c) {
              const uint64_t s2 = s20;  // chunks 0-3: gate columns (mode 0) / first weight-scale block
  #pragma unroll
              for (int i = 0; i < 16; i += 2) ptx::fma2(acc2[c * 8 + i / 2], v[c][i], v[c][i + 1], s2);
              ptx::tmem_ld16(tb + (c + 4) * 16, v[c]);
            }
            ptx::tmem_ld_wait16(v[0]);
            ptx::keep16(v[1]); ptx::keep16(v[2]); ptx::keep16(v[3]);
            // the whole partial is in registers: hand the TMEM buffer back before the last FMAs
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              if (kPair && rank != 0) ptx::mbar_arrive_cluster(te_a + 8 * buf);  // remote: the leader's barrier
              else ptx::mbar_arrive_a(bar_a + kOffTmemEmpty + 8 * buf);
            }
  #pragma unroll
            for (int c = 0; c < 4; ++c) {
              const uint64_t s2 = s21;  // chunks 4-7: up columns (mode 0) / same block (mode 1: s21 == s20)
  #pragma unroll
              for (int i = 0; i < 16; i += 2) ptx::fma2(acc2[(c + 4) * 8 + i / 2], v[c][i], v[c][i + 1], s2);
            }
          }
          ++it;
        }
      }
#ifdef SLP_PROF
      const long long p2 = clock64();
#endif
      if (has_next) open_tile(nx);  // first scale loads of the next tile fly during this tile's epilogue
      float acc[128];
#pragma unroll
      for (int i = 0; i < 64; ++i) ptx::unpack2(acc2[i], acc[2 * i], acc[2 * i + 1]);

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
        ptx::named_bar_sync(1 + q, 64);  // only the two warps that share these 32 rows (w and w + 4) meet
        amax = fmaxf(amax, ex[(half ^ 1) * BM + r_in_tile]);
        const float s = (amax == 0.f) ? 1.0f : __fdiv_rn(amax, 448.0f);
        if (row_ok_cur) {
          // e4m3(h / s) with IEEE division semantics from one reciprocal + a residual step (div_by).  A
          // denormal-range scale (never seen on real activations) is handled by scaling h and s by 2^64
          // first, which is exact and leaves every quotient unchanged.
          float sq = s;
          if (s < 1e-30f) {
            sq = s * 0x1p64f;
#pragma unroll
            for (int i = 0; i < 64; ++i) acc[i] *= 0x1p64f;
          }
          const float r = __frcp_rn(sq);
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) pk[i] = quant4_e4m3_r(acc[4 * i], acc[4 * i + 1], acc[4 * i + 2], acc[4 * i + 3], sq, r);
          uint4* dst = reinterpret_cast<uint4*>(g.hq + row * g.I + nt * 128 + half * 64);
#pragma unroll
          for (int i = 0; i < 4; ++i) dst[i] = make_uint4(pk[4 * i], pk[4 * i + 1], pk[4 * i + 2], pk[4 * i + 3]);
          if (half == 0) g.hs[row * g.hs_stride + nt] = s;
        }
      } else {
        // Y tile, stored as block-scaled fp16: a thread owns one row x 128 columns, exactly one scale block.
        // It takes the block's amax, scales by the power of two that puts amax into [2^14, 2^15) (exact),
        // rounds to fp16 (10-bit mantissa: 2^-11 relative, an eighth of a bf16 step, with fp32's range
        // through the per-block exponent; DESIGN.md 3.4 has the error budget) and writes the scale 2^e to
        // ys[row, block].  Each warp's 32 rows x 128 columns = two 32 x 64 boxes (128-byte rows, 128B
        // swizzle: conflict-free st.shared.v4, whole-line global writes).  The whole tile fits in the
        // staging area, so the warp writes both boxes, hands them to TMA stores and starts the next tile's
        // K loop without waiting for a free slot; the boxes of the previous tile were read out long ago
        // (16 K blocks), the wait below is a formality.  Rows past the expert's count are padding rows of
        // the workspace; whole 32-row groups past it are skipped.
        const int c0 = nt * BN + half * HN;
        if (c0 < g.H && q * 32 < nrows) {
          float am[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};  // eight independent chains instead of one of 128
#pragma unroll
          for (int i = 0; i < 128; i += 16) {
#pragma unroll
            for (int u = 0; u < 8; ++u) am[u] = fmaxf(am[u], fmaxf(fabsf(acc[i + 2 * u]), fabsf(acc[i + 2 * u + 1])));
          }
          const float amax = fmaxf(fmaxf(fmaxf(am[0], am[1]), fmaxf(am[2], am[3])), fmaxf(fmaxf(am[4], am[5]), fmaxf(am[6], am[7])));
          const uint32_t eb = max(__float_as_uint(amax) >> 23, 14u);          // biased exponent of amax (>= 0)
          const float mult = __uint_as_float((268u - eb) << 23);                // 2^(14 - floor(log2 amax))
          g.ys[row * g.ys_stride + (c0 >> 7)] = __uint_as_float((eb - 14u) << 23);  // 2^(floor(log2 amax) - 14)
          const uint32_t stage_a = smem_a + kStages * kStageBytes + warp * 8192;
          const uint32_t sw = static_cast<uint32_t>(lane & 7);
          if (lane == 0) ptx::bulk_wait_group_read<0>();
          __syncwarp();
#pragma unroll
          for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const float* a8 = acc + c * 64 + j * 8;
              const uint32_t dst = stage_a + c * 4096 + lane * 128 + ((static_cast<uint32_t>(j) ^ sw) << 4);
              asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "r"(ptx::pack_f16x2(a8[0] * mult, a8[1] * mult)),
                           "r"(ptx::pack_f16x2(a8[2] * mult, a8[3] * mult)), "r"(ptx::pack_f16x2(a8[4] * mult, a8[5] * mult)),
                           "r"(ptx::pack_f16x2(a8[6] * mult, a8[7] * mult)) : "memory");
            }
          }
          ptx::fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            ptx::tma_store_2d_a(&tm_y, stage_a, c0, row0 + q * 32);
            ptx::tma_store_2d_a(&tm_y, stage_a + 4096, c0 + 64, row0 + q * 32);
            ptx::bulk_commit_group();
          }
        }
      }
#ifdef SLP_PROF
      { const long long p3 = clock64(); pf += p1 - pa; pq += pa - p0; pk += p2 - p1; pe += p3 - p2; pn += 1; }
#endif
    }
#ifdef SLP_PROF
    if (warp == 0 && lane == 0) {
      atomicAdd(&g.clk[4 + 4 * kMode], static_cast<unsigned long long>(pf));
      atomicAdd(&g.clk[5 + 4 * kMode], static_cast<unsigned long long>(pk));
      atomicAdd(&g.clk[6 + 4 * kMode], static_cast<unsigned long long>(pe));
      atomicAdd(&g.clk[7 + 4 * kMode], static_cast<unsigned long long>(pn));
      atomicAdd(&g.clk[12 + kMode], static_cast<unsigned long long>(pq));
    }
#endif
    if (kMode == 1 && lane == 0) ptx::bulk_wait_group_read<0>();  // staging memory must outlive the last stores
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long ns1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns1));
    atomicAdd(&g.clk[2 * kMode], static_cast<unsigned long long>(clock64() - clk0));
    atomicAdd(&g.clk[2 * kMode + 1], ns1 - ns0);
  }
  if (kPair) ptx::cluster_sync();  // no CTA leaves while its peer can still signal its barriers or read its smem
  if (warp == kEpiWarps + 1) {
    ptx::tc_fence_after();
    if (kPair) ptx::tmem_dealloc_2sm<kTmemCols>(tmem_base);
    else ptx::tmem_dealloc<kTmemCols>(tmem_base);
  }
}

}  // namespace tc
}  // namespace slp
