// kernels_gemm_tc.cuh — grouped FP8 GEMM on the 5th-gen tensor cores (a5, a6, a7, a8).
//
// One persistent CTA per SM works through the (128-row tile, N tile) work items of the experts of the
// launch (one 16-byte record per tile, written by permute_scan_kernel); an otherwise idle warp takes the
// items from a global counter, so all CTAs stay within ~gridDim consecutive items and share operands
// through L2 (triage "gemm=static": static round-robin instead).  Per 128-deep K block the tensor core
// writes a fresh 128 x 256 fp32 partial into TMEM, as two independent 128-column halves (four half-buffers
// in flight); the promotion warps pull it out with tcgen05.ld and add it into fp32 register accumulators
// with one FMA per element (issued as FFMA2 pairs), scaled by  xs[row, kb] * ws[n-block, kb]
// ("FP8 GEMM with FP32 accumulation"; "accumulate all partial dot-products
// first and apply the scale once per block").
//
//   warp 8      TMA producer (one elected thread): A tile (128 rows x 128 B) + 64-row B boxes per K
//               block into a 128B-swizzled smem ring (mbarrier full / empty)
//   warp 9      MMA issuer (one elected thread): per K block and column half 4 x tcgen05.mma.kind::f8f6f4
//               (M128 N128 K32) into TMEM half-buffer [kb mod 2][half]; tcgen05.commit publishes the
//               half-buffer, a last commit frees the stage; its three barrier probes per K block are in
//               flight together
//   warp 10     work scheduler (one elected thread): atomicAdd on the launch's counter, reads the tile's
//               record and publishes it through a 4-deep smem ring read by the producer, the MMA issuer
//               and the promotion warps
//   warp 11     idle (warps 8-11 donate most of their registers to the promotion warps, setmaxnreg)
//   warps 0-7   promotion + epilogue: warp w owns TMEM lanes 32 * (w % 4).. (rows) and the 128 columns
//               of half w / 4; 128 fp32 accumulators per thread; a half-buffer is handed back as soon as
//               the last tcgen05.ld has landed, before the last FMAs
//
// kPair (triage "gemm=pair"): a cluster of two CTAs issues cta_group::2 MMAs with M = 256 (two
//   128-row tiles of the same expert) x N = 128 per column half; each CTA stages its own A tile and half of
//   the B tile (CTA 0 the gate rows / CTA 1 the up rows of a gate/up tile; 64 rows of each column half of a
//   down tile); TMA loads of both CTAs complete on the leader's mbarrier, commits are multicast to both CTAs,
//   the peer's promotion warps release TMEM on the leader's barrier.  It moves a third less operand data
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
constexpr int kWsCap = 64;      // K blocks of weight scales a promotion warp keeps in shared memory (refilled beyond)

// kPair = false: one CTA per tile, A tile (16 KB) + whole B tile (32 KB) per stage, 4 stages.
// kPair = true:  a cluster of two CTAs issues one cta_group::2 MMA with M = 256 (two 128-row tiles
//                of the same expert) x N = 256; each CTA stages its own A tile and HALF of the B tile
//                (16 KB + 16 KB per stage, 6 stages), which cuts the L2 -> SM operand traffic per MAC
//                by a third (the 1-CTA kernel is L2-bandwidth bound, profiles/r1_gemm_baseline.md).
template <int kMode, bool kPair> struct Cfg {
  // The down kernel trades one pipeline stage for a staging area that holds its whole fp16 Y tile
  // (64 KB): its tiles are only 16 K blocks long, so the epilogue must not wait on TMA-store read-out.
  static constexpr int kStages = kPair ? (kMode == 1 ? 4 : 6) : (kMode == 1 ? 3 : 4);
  static constexpr int kABytes = BM * BK;
  static constexpr int kBBytes = (kPair ? BN / 2 : BN) * BK;
  static constexpr int kStageBytes = kABytes + kBBytes;
  // mode 1: the whole fp16 Y tile (two 4 KB boxes per warp); mode 0: the amax exchange (2 KB); both: the per-warp
  // weight-scale tables of the promotion loop (kWsCap float2 per warp)
  static constexpr int kYBytes = kMode == 1 ? kEpiWarps * 8192 : 2048;
  static constexpr int kScratchBytes = kYBytes + kEpiWarps * kWsCap * 8;
  static constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 512 /*barriers*/ + kScratchBytes;
  static_assert(kSmemBytes <= 232448, "shared memory budget");
};

// Barrier block behind the stage ring; the kernels address it through 32-bit shared addresses.
struct Shared {
  uint64_t full[kMaxStages];   // TMA -> MMA: stage landed (pair: lives in the leader CTA, fed by both CTAs' loads)
  uint64_t empty[kMaxStages];  // MMA -> TMA: stage consumed (pair: multicast commit to both CTAs)
  uint64_t tmem_full[2][2];    // MMA -> promotion: columns [128 h, 128 h + 128) of the K block partial complete in TMEM buffer b: [b][h]
  uint64_t tmem_empty[2][2];   // promotion -> MMA: that half of buffer b read out by its kEpiWarps / 2 warps (pair: both CTAs', at the leader)
  uint64_t sched_full[kSchedDepth];   // scheduler -> roles: work item published
  uint64_t sched_empty[kSchedDepth];  // roles -> scheduler: slot read by producer, MMA issuer and the promotion warps
  int4 sched_rec[kSchedDepth];        // tile record of each slot {expert (-1 = no more work), first row, valid rows, N tile}
  uint32_t tmem_base;
  int dead;
};
static_assert(sizeof(Shared) <= 512, "barrier block");
constexpr uint32_t kOffFull = 0, kOffEmpty = 8 * kMaxStages, kOffTmemFull = 16 * kMaxStages, kOffTmemEmpty = 16 * kMaxStages + 32;
constexpr uint32_t kOffSchedFull = kOffTmemEmpty + 32, kOffSchedEmpty = kOffSchedFull + 8 * kSchedDepth;

// silu(g) * u for two elements with the fast exponential and ONE reciprocal (rel. error ~1e-6, three decades below
// the e4m3 step that follows): 1 / a = b * rcp(a b), 1 / b = a * rcp(a b) with a = 1 + e^-g0, b = 1 + e^-g1.  The SFU
// (16 results per clock per SM) bounds this epilogue, so three instead of four SFU operations per pair matter.
// e^-g is clamped to 2^60 so that the product stays finite (silu(g) < 2^-54 there anyway).
__device__ __forceinline__ void silu_mul_fast2(float& g0, float u0, float& g1, float u1) {
  float t0, t1, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(t0) : "f"(g0 * -1.4426950408889634f));
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(t1) : "f"(g1 * -1.4426950408889634f));
  const float a = 1.0f + fminf(t0, 0x1p60f), b = 1.0f + fminf(t1, 0x1p60f);
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a * b));
  g0 = g0 * (r * b) * u0;
  g1 = g1 * (r * a) * u1;
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
    for (int i = 0; i < 4; ++i) { ptx::mbar_init(&sh->tmem_full[i >> 1][i & 1], 1); ptx::mbar_init(&sh->tmem_empty[i >> 1][i & 1], kPair ? kEpiWarps : kEpiWarps / 2); }
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

  // Tile that follows this CTA's i-th one (e < 0: none).  Static order: item w + gridDim, record read from global
  // memory.  kDyn (one-CTA kernel, the default; triage "gemm=static" selects the static order): items come from a
  // global counter, so all CTAs stay inside a window of ~gridDim consecutive items and the B tiles they share stay in
  // L2 (profiles/r1_sched_ab.md).  An otherwise idle warp takes the item AND reads its record, and publishes the
  // record through a four-deep ring in shared memory: the roles pay one barrier wait and one 16-byte shared load per
  // tile instead of a global-memory round trip (a record held in registers across the K loop was being spilled and
  // cost the promotion warps ~650 cycles per tile).  Which CTA computes a tile does not change its result.
  const uint32_t rec_a = bar_a + static_cast<uint32_t>(offsetof(Shared, sched_rec));
  auto next_tile = [&](int& w, int i, bool whole_warp) -> Tile {
    Tile t;
    if constexpr (kPair || !kDyn) {
      w += w_step;
      if (w < total) t = fetch(w);
      else t.e = -1;
    } else {
      const uint32_t slot = static_cast<uint32_t>(i) % kSchedDepth;
      ptx::mbar_wait_a(bar_a + kOffSchedFull + 8 * slot, (static_cast<uint32_t>(i) / kSchedDepth) & 1, dead, g.err, 5);
      const int4 r = ptx::lds_s32x4(rec_a + 16 * slot);  // warp-uniform address
      t.e = r.x; t.row0 = r.y; t.nrows = r.z; t.nt = r.w;
      if (whole_warp) {
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_a(bar_a + kOffSchedEmpty + 8 * slot);
      } else {
        ptx::mbar_arrive_a(bar_a + kOffSchedEmpty + 8 * slot);
      }
    }
    return t;
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
      Tile nx{-1, 0, 0, 0};
      if (w_first < total) nx = fetch(w_first);  // idle CTAs (and launches without any tile) read no record
      int w = w_first;
      for (int i = 0; nx.e >= 0; ++i) {
        const Tile cur = nx;
        nx = next_tile(w, i, false);
        const int e = cur.e, nt = cur.nt, row0 = cur.row0;
        const int slot = slot_of(g, e);
        constexpr int kBoxes = kPair ? 2 : 4;
        int brow[kBoxes];
        if (kMode == 0) {
          // pool = [gate of all slots | up of all slots | down of all slots], viewed as [3 * slots * I, H]
          const int gate0 = slot * g.I + nt * 128, up0 = (g.n_slots + slot) * g.I + nt * 128;
          if (kPair) { brow[0] = rank == 0 ? gate0 : up0; brow[1] = brow[0] + 64; }  // CTA 0: gate rows, CTA 1: up rows (64 per column half)
          else { brow[0] = gate0; brow[1] = up0; brow[2 % kBoxes] = gate0 + 64; brow[3 % kBoxes] = up0 + 64; }
        } else {
          const int down0 = (2 * g.n_slots + slot) * g.H + nt * BN;  // same pool viewed as [3 * slots * H, I]
          if (kPair) { brow[0] = down0 + 64 * rank; brow[1] = brow[0] + 128; }  // 64 rows of each column half
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
        int4 r = make_int4(-1, 0, 0, 0);
        if (w < total) {
          const Tile t = fetch(w);
          r = make_int4(t.e, t.row0, t.nrows, t.nt);
        }
        ptx::sts_s32x4(rec_a + 16 * slot, r);
        ptx::mbar_arrive_a(bar_a + kOffSchedFull + 8 * slot);  // release: the store above is visible to the waiters
        if (w >= total) break;
      }
    }
   } else if (warp == kEpiWarps + 1) {
    // ===================== MMA issuer (one elected thread; pair: leader CTA only) =====================
    if (rank == 0 && ptx::elect_one()) {
      // A K block is issued as two N = 128 MMAs groups (columns [0, 128) and [128, 256) of the tile) with their own
      // TMEM hand-off barriers: four 128-column buffers are in flight instead of two 256-column ones, so a half
      // buffer has three MMA groups (768 cycles) to be drained and handed back before the tensor core needs it again,
      // and the two promotion warps that share a scheduler work 256 cycles apart instead of in lock step.  Price: the
      // A tile is read from shared memory twice per K block.
      constexpr uint32_t idesc = ptx::umma_idesc_e4m3_f32(kPair ? 2 * BM : BM, HN);
      constexpr uint64_t kHalfB = (kPair ? HN / 2 : HN) * BK / 16;  // B rows of column half 1 start here (16-byte units)
      const uint64_t adesc0 = ptx::umma_desc_k128_a(smem_a), bdesc0 = ptx::umma_desc_k128_a(smem_a + kABytes);
      int stage = 0;
      uint32_t phase = 0;
      uint32_t it = 0;  // running K-block counter: TMEM buffer = it & 1
      int w = w_first;
      bool have = w_first < total;
      for (int i = 0; have; have = next_tile(w, i, false).e >= 0, ++i) {
        for (int kb = 0; kb < num_kb; ++kb, ++it) {
          const uint32_t buf = it & 1, tph = ((it >> 1) & 1) ^ 1;
          // A barrier probe takes ~100 cycles to answer even when the phase completed long ago, and this one thread
          // needs three answers per K block: the three probes are issued back to back (test_wait never suspends the
          // thread) and only a phase that is still open is then waited for.  Waiting for them one after the other made
          // this loop, not the tensor core, the bound of the kernel (~500 cycles per K block).
          const uint32_t fa = bar_a + kOffFull + 8 * stage, e0a = bar_a + kOffTmemEmpty + 16 * buf, e1a = e0a + 8;
          const bool pf = ptx::mbar_test_wait_a(fa, phase);
          const bool p0 = ptx::mbar_test_wait_a(e0a, tph);
          const bool p1 = ptx::mbar_test_wait_a(e1a, tph);
          if (!pf) ptx::mbar_wait_a(fa, phase, dead, g.err, 3);   // operands landed (usually long ago)
          const uint64_t so = static_cast<uint64_t>((stage * kStageBytes) >> 4);
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (!(h == 0 ? p0 : p1)) ptx::mbar_wait_a(h == 0 ? e0a : e1a, tph, dead, g.err, 2);   // the hand-off: issue right after it
            ptx::tc_fence_after();
            const uint32_t d = tmem_base + buf * BN + h * HN;
#pragma unroll
            for (int k4 = 0; k4 < BK / 32; ++k4) {  // UMMA_K = 32 for 8-bit operands: +32 B per step
              if (kPair) ptx::umma_f8_2sm(d, adesc0 + so + 2 * k4, bdesc0 + so + h * kHalfB + 2 * k4, idesc, k4 > 0);
              else ptx::umma_f8(d, adesc0 + so + 2 * k4, bdesc0 + so + h * kHalfB + 2 * k4, idesc, k4 > 0);
            }
            if (kPair) ptx::umma_commit_2sm_mc(bar_a + kOffTmemFull + 16 * buf + 8 * h, 3);  // both CTAs' rows of this half are complete
            else ptx::umma_commit_a(bar_a + kOffTmemFull + 16 * buf + 8 * h);
          }
          if (kPair) ptx::umma_commit_2sm_mc(bar_a + kOffEmpty + 8 * stage, 3);   // both CTAs' stages reusable once these MMAs retire
          else ptx::umma_commit_a(bar_a + kOffEmpty + 8 * stage);
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
    const uint32_t te_a = lead_bar + kOffTmemEmpty + 8 * half;  // [buffer][this warp's column half]; pair: the leader's barrier (cluster address)
    const uint32_t tf_a = bar_a + kOffTmemFull + 8 * half;
    // Per-tile scales.  The row's activation scales xs[row, kb] come as one 16-byte load per four K blocks (issued
    // four K blocks ahead); the weight scales (ws0[kb], ws1[kb]) of the tile go through a small per-warp table in
    // shared memory: lane l fetches K blocks l and l + 32 while the previous tile's epilogue runs, the table is
    // written at the start of the K loop and every K block costs one 8-byte shared load at a warp-uniform address.
    const float *as_ptr = nullptr, *ws0 = nullptr, *ws1 = nullptr;
    bool row_ok = false;
    float4 xs_nxt = make_float4(0.f, 0.f, 0.f, 0.f);
    float wa0 = 0.f, wa1 = 0.f, wb0 = 0.f, wb1 = 0.f;  // prefetched weight scales: K blocks lane (a) and lane + 32 (b)
    const uint32_t wsm_a = ptx::launder_u32(smem_a + kStages * kStageBytes + C::kYBytes + warp * (kWsCap * 8));  // this warp's table
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
      xs_nxt = row_ok ? *reinterpret_cast<const float4*>(as_ptr) : make_float4(0.f, 0.f, 0.f, 0.f);
      wa0 = lane < num_kb ? ws0[lane] : 0.f;
      wb0 = lane + 32 < num_kb ? ws0[lane + 32] : 0.f;
      if (kMode == 0) {
        wa1 = lane < num_kb ? ws1[lane] : 0.f;
        wb1 = lane + 32 < num_kb ? ws1[lane + 32] : 0.f;
      }
    };
    // weight scales of K blocks [k0, k0 + kWsCap) of the open tile -> table (k0 > 0 only when num_kb > kWsCap)
    auto refill_ws = [&](int k0) {
      __syncwarp();
      for (int k = lane; k < kWsCap; k += 32) {
        const int kk = k0 + k;
        ptx::sts_f32x2(wsm_a + 8 * k, kk < num_kb ? ws0[kk] : 0.f, (kMode == 0 && kk < num_kb) ? ws1[kk] : 0.f);
      }
      __syncwarp();
    };
    Tile nx{-1, 0, 0, 0};
    if (w_first < total) { nx = fetch(w_first); open_tile(nx); }
    int w = w_first;
#ifdef SLP_PROF
    long long pk = 0, pe = 0, pf = 0, pn = 0, pq = 0;
#endif
    for (int ti = 0; nx.e >= 0; ++ti, tile_parity ^= 1) {
      const Tile cur = nx;
#ifdef SLP_PROF
      const long long pa = clock64();
      long long p1 = pa;
#endif
      const int nt = cur.nt, row0 = cur.row0, nrows = cur.nrows;
      const size_t row = static_cast<size_t>(row0 + r_in_tile);
      const bool row_ok_cur = row_ok;
      float acc[128];  // fp32 accumulators, updated in FFMA2 pairs
#pragma unroll
      for (int i = 0; i < 128; ++i) acc[i] = 0.f;
      __syncwarp();  // every lane is done reading the previous tile's table
      ptx::sts_f32x2(wsm_a + 8 * lane, wa0, wa1);
      ptx::sts_f32x2(wsm_a + 8 * (lane + 32), wb0, wb1);
      __syncwarp();

      // One K block: the warp waits for the partial of ITS column half in TMEM buffer it & 1 (the MMA issuer
      // publishes the two 128-column halves of a K block separately, see there), pulls the thread's 128 columns out
      // in 8 chunks of 16 through four register sets and adds them, scaled, into the accumulators.  Chunks 0-3 are
      // requested up front, chunk c + 4 as soon as the FMAs of chunk c have consumed its set, so every tcgen05.ld of
      // the K block has landed after half of the FMAs and the half-buffer goes back to the MMA issuer there.
      auto k_block = [&](float sa, int kb) {
        const float2 wsc = ptx::lds_f32x2(wsm_a + 8 * (kb & (kWsCap - 1)));  // warp-uniform address; lands during the wait below
        const uint32_t buf = it & 1;
        ptx::mbar_wait_a(tf_a + 16 * buf, (it >> 1) & 1, dead, g.err, 4);
        ptx::tc_fence_after();
#ifdef SLP_PROF
        if (kb == 0) p1 = clock64();
#endif
        const uint32_t tb = tm_lane + buf * BN;
        uint32_t v[4][16];
#pragma unroll
        for (int c = 0; c < 4; ++c) ptx::tmem_ld16(tb + c * 16, v[c]);
        const float sc0 = sa * wsc.x;                           // gate columns (mode 0) / the one weight-scale block (mode 1)
        const float sc1 = kMode == 0 ? sa * wsc.y : sc0;        // up columns (mode 0)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
#pragma unroll
          for (int i = 0; i < 16; i += 2) ptx::fma2f(acc[c * 16 + i], acc[c * 16 + i + 1], v[c][i], v[c][i + 1], sc0);
          ptx::tmem_ld16(tb + (c + 4) * 16, v[c]);
        }
        ptx::tmem_ld_wait();
        // the whole partial is in registers: hand the TMEM half-buffer back before the last FMAs
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          if (kPair && rank != 0) ptx::mbar_arrive_cluster(te_a + 16 * buf);  // remote: the leader's barrier
          else ptx::mbar_arrive_a(te_a + 16 * buf);
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
#pragma unroll
          for (int i = 0; i < 16; i += 2) ptx::fma2f(acc[(c + 4) * 16 + i], acc[(c + 4) * 16 + i + 1], v[c][i], v[c][i + 1], sc1);
        }
        ++it;
      };

#pragma unroll 1
      for (int kb0 = 0; kb0 < num_kb; kb0 += 4) {
        if (kb0 != 0 && (kb0 & (kWsCap - 1)) == 0) refill_ws(kb0);
        const float4 xs4 = xs_nxt;
        if (kb0 + 4 < num_kb && row_ok) xs_nxt = *reinterpret_cast<const float4*>(as_ptr + kb0 + 4);
        k_block(xs4.x, kb0);
        if (kb0 + 1 < num_kb) k_block(xs4.y, kb0 + 1);
        if (kb0 + 2 < num_kb) k_block(xs4.z, kb0 + 2);
        if (kb0 + 3 < num_kb) k_block(xs4.w, kb0 + 3);
      }
#ifdef SLP_PROF
      const long long p2 = clock64();
#endif
#ifdef SLP_PROF
      const long long q0 = clock64();
#endif
      nx = next_tile(w, ti, true);   // one barrier wait + one 16-byte shared load (the scheduler warp read the record)
      if (nx.e >= 0) open_tile(nx);  // first scale loads of the next tile fly during this tile's epilogue
#ifdef SLP_PROF
      pq += clock64() - q0;
#endif

      if (kMode == 0) {
        // h = silu(gate) * up over this thread's 64 channels; row amax over all 128 via smem
        float amax = 0.f;
#pragma unroll
        for (int i = 0; i < 64; i += 2) {
          silu_mul_fast2(acc[i], acc[64 + i], acc[i + 1], acc[64 + i + 1]);
          amax = fmaxf(amax, fmaxf(fabsf(acc[i]), fabsf(acc[i + 1])));
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
      { const long long p3 = clock64(); pf += p1 - pa; pk += p2 - p1; pe += p3 - p2; pn += 1; }
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
