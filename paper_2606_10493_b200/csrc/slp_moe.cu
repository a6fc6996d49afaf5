// slp_moe.cu — host side of libslpmoe: handle, C ABI (include/slp_moe.h), workspace, TMA
// descriptors and the streaming engine (a4) that overlaps host->HBM expert-weight copies with the
// grouped GEMMs (Fig. 5: loader / model / unloader with ON / OFF events and an
// experts ring buffer).  On one device the three roles collapse to two CUDA streams and two event
// arrays: the copy stream is the loader, the caller's stream is the model thread, and "unload" is
// the slot-free event the loader waits on before it overwrites a ring slot (the authoritative copy
// stays on the host, so nothing is copied back).
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/slp_moe.h"
#include "kernels_gemm_simt.cuh"
#include "kernels_gemm_tc.cuh"
#include "kernels_route.cuh"
#include "kernels_router_tc.cuh"

namespace {

thread_local std::string g_last_error;

slp_status fail(slp_status st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_last_error = buf;
  return st;
}

#define CU_TRY(expr)                                                                                   \
  do {                                                                                                 \
    cudaError_t _e = (expr);                                                                           \
    if (_e != cudaSuccess) {                                                                           \
      slp_status _st = (_e == cudaErrorMemoryAllocation) ? SLP_ERR_OOM : SLP_ERR_CUDA;                 \
      return fail(_st, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__);    \
    }                                                                                                  \
  } while (0)

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  return fn;
}

// 2D uint8 tensor [rows, inner] (row stride = inner bytes), box 128 B x box_rows rows, 128B swizzle.
slp_status make_tmap_u8(CUtensorMap* tm, void* base, uint64_t inner, uint64_t rows, uint32_t box_rows = 128) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return fail(SLP_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");
  cuuint64_t dims[2] = {inner, rows};
  cuuint64_t strides[1] = {inner};
  cuuint32_t box[2] = {128, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(SLP_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", static_cast<int>(r));
  return SLP_OK;
}

// 2D fp16 tensor [rows, inner] for TMA stores of 64-column x 32-row boxes (128-byte rows, 128B swizzle).
slp_status make_tmap_f16_store(CUtensorMap* tm, void* base, uint64_t inner, uint64_t rows) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return fail(SLP_ERR_CUDA, "cuTensorMapEncodeTiled not available from the driver");
  cuuint64_t dims[2] = {inner, rows};
  cuuint64_t strides[1] = {inner * 2};
  cuuint32_t box[2] = {64, 32};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(SLP_ERR_CUDA, "cuTensorMapEncodeTiled (Y store) failed with CUresult %d", static_cast<int>(r));
  return SLP_OK;
}

// experts_per_launch = 0 (auto): up to 64 experts per grouped-GEMM launch when the ring holds the
// whole layer (amortises the launch ramp and tail: 0.40 -> 0.70 of the HBM roofline on the T = 4096
// layer, while the host-link-bound step moves by < 0.1 %); a ring shorter than the layer needs a
// divisor of the ring length that is at most half of it (and at most 32).
inline int auto_epl(int n_stage, int E) {
  if (n_stage == E) return std::min(64, E);
  int best = 1;
  for (int d = 1; d <= std::min(32, n_stage / 2); ++d)
    if (n_stage % d == 0) best = d;
  return best;
}

constexpr int kTailExperts = 8;  // experts per launch inside the last launch group of a streamed call (prefill_impl)

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// Triage switches (not a product option): bring-up / A-B variants of two kernels, so a wrong result can be bisected
// on a GPU box without rebuilding.  They are handed over per thread through slp_moe_debug_set_triage() and consumed by
// the next create on that thread; the library reads no environment variable, so nothing in a process's environment can
// change which kernels a handle runs.  Comma-separated tokens:
//   gemm=simt    plain CUDA-core grouped GEMM (kernels_gemm_simt.cuh) instead of the tcgen05 kernels
//   gemm=static  one-CTA tcgen05 kernel with the static round-robin tile order
//   gemm=pair    the cta_group::2 variant of the tcgen05 kernel
//   router=fp32  router logits as plain fp32 FMAs instead of the tensor-core hi/lo split
//   guards       every workspace buffer gets a 4 KB canary band before and after it; slp_moe_get_stats and destroy
//                fail with SLP_ERR_CUDA if a band was written (compute-sanitizer is closed on the GPU pool);
//                guards=selftest additionally writes one byte behind the counts buffer at create
enum GemmImpl { kGemmTc = 0, kGemmSimt = 1, kGemmPair = 2, kGemmStatic = 3 };
struct Triage {
  int gemm = kGemmTc;
  int router_fp32 = 0;
  int guards = 0;
};
thread_local Triage g_triage_next;  // what the next create on this thread takes (default: the product path)

// Parses a triage spec; false (and *bad = the offending token) on an unknown token.
bool parse_triage(const std::string& v, Triage* t, std::string* bad) {
  size_t pos = 0;
  while (pos <= v.size()) {
    size_t end = v.find(',', pos);
    if (end == std::string::npos) end = v.size();
    const std::string tok = v.substr(pos, end - pos);
    if (tok.empty()) {}
    else if (tok == "gemm=simt") t->gemm = kGemmSimt;
    else if (tok == "gemm=static") t->gemm = kGemmStatic;
    else if (tok == "gemm=pair") t->gemm = kGemmPair;
    else if (tok == "router=fp32") t->router_fp32 = 1;
    else if (tok == "guards") t->guards = std::max(t->guards, 1);
    else if (tok == "guards=selftest") t->guards = 2;  // create damages one band on purpose (negative control)
    else { *bad = tok; return false; }
    pos = end + 1;
  }
  return true;
}

inline Triage read_triage() {
  const Triage t = g_triage_next;
  g_triage_next = Triage{};
  return t;
}

// Shape / option validation shared by create and slp_moe_query_plan (no CUDA calls).  On success
// *n_stage = expert slots of the streamed ring, *epl = experts per grouped-GEMM launch.
slp_status validate_cfg(const slp_moe_cfg* cfg, int* n_stage_out, int* epl_out) {
  const int H = cfg->hidden, E = cfg->n_experts, k = cfg->top_k, I = cfg->moe_intermediate, G = cfg->n_group, Gk = cfg->topk_group;
  if (H <= 0 || I <= 0 || H % 128 || I % 128 || H / 128 > 1024 || I / 128 > 1024)
    return fail(SLP_ERR_UNSUPPORTED_SHAPE, "hidden (%d) and moe_intermediate (%d) must be positive multiples of 128", H, I);
  if (E <= 0 || E > slp::kMaxExperts - 1) return fail(SLP_ERR_UNSUPPORTED_SHAPE, "n_experts %d outside 1..%d", E, slp::kMaxExperts - 1);
  if (G <= 0 || G > 32 || E % G || Gk <= 0 || Gk > G) return fail(SLP_ERR_UNSUPPORTED_SHAPE, "n_group %d / topk_group %d invalid for %d experts", G, Gk, E);
  if (k <= 0 || k > 32 || k > E || static_cast<long long>(k) > static_cast<long long>(Gk) * (E / G))
    return fail(SLP_ERR_UNSUPPORTED_SHAPE, "top_k %d invalid (needs 1..32, <= topk_group * E / n_group)", k);
  if (cfg->n_shared < 0 || cfg->n_shared > 1 || (cfg->n_shared == 1 && cfg->shared_intermediate != I))
    return fail(SLP_ERR_UNSUPPORTED_SHAPE, "n_shared must be 0 or 1 with shared_intermediate == moe_intermediate");
  if (cfg->scoring != SLP_SCORE_SIGMOID_BIAS && cfg->scoring != SLP_SCORE_SOFTMAX) return fail(SLP_ERR_INVALID_ARG, "unknown scoring %d", cfg->scoring);
  if (cfg->max_tokens <= 0) return fail(SLP_ERR_INVALID_ARG, "max_tokens must be positive");
  if (cfg->expert_begin < 0 || cfg->expert_end < 0 || cfg->expert_end > E || (cfg->expert_end != 0 && cfg->expert_begin >= cfg->expert_end) ||
      (cfg->expert_end == 0 && cfg->expert_begin != 0))
    return fail(SLP_ERR_INVALID_ARG, "expert range [%d, %d) invalid for %d experts (0, 0 = all)", cfg->expert_begin, cfg->expert_end, E);
  const int En = cfg->expert_end == 0 ? E : cfg->expert_end - cfg->expert_begin;  // experts this handle owns
  int n_stage = cfg->staging_slots == 0 ? En : cfg->staging_slots;
  if (n_stage < 2 && En >= 2) return fail(SLP_ERR_INVALID_ARG, "staging_slots must be 0 or 2..(owned experts)");
  n_stage = std::min(n_stage, En);
  int epl = cfg->experts_per_launch;
  if (epl == 0) epl = auto_epl(n_stage, En);
  if (epl < 1 || epl > n_stage || (n_stage != En && (epl > n_stage / 2 || n_stage % epl)))
    return fail(SLP_ERR_INVALID_ARG, "experts_per_launch %d invalid for %d staging slots (must divide it, <= half)", epl, n_stage);
  *n_stage_out = n_stage;
  *epl_out = epl;
  return SLP_OK;
}

}  // namespace

// Everything that belongs to ONE layer of a stack: host pointers and the small resident tensors.  The handle
// keeps the set of the layer it is working on in its own fields of the same names (select_layer).
struct LayerW {
  slp_moe_host_weights hw{};
  std::vector<const uint8_t*> gate_q, up_q, down_q;
  uint16_t* d_router_hl = nullptr;
  CUtensorMap tm_rw{};
  float *d_router_w = nullptr, *d_bias = nullptr, *d_gate_s = nullptr, *d_up_s = nullptr, *d_down_s = nullptr;
  uint8_t* d_shpool = nullptr;  // [3][I*H] shared expert of layers > 0 (layer 0's sits in slot 0 of the ring pool)
  CUtensorMap tm_shgu{}, tm_shd{};
};

struct slp_moe_layer {
  slp_moe_cfg cfg{};
  Triage triage{};
  std::vector<LayerW> layers;  // n_layers weight sets sharing one ring, one workspace
  int cur_layer = -1;
  // ring occupancy, per ring group: which (layer, first expert) was loaded into it last, and whether that load
  // was a prefetch nobody has consumed yet (the loader running ahead of the model thread)
  std::vector<int> occ_layer, occ_e0;
  std::vector<char> occ_prefetched;
  slp_moe_host_weights hw{};
  std::vector<const uint8_t*> gate_q, up_q, down_q;
  uint8_t* d_shpool = nullptr;
  CUtensorMap tm_shgu{}, tm_shd{};
  std::vector<void*> registered;  // host ranges pinned by create
  int H = 0, E = 0, k = 0, I = 0, Tm = 0;
  int e0 = 0, e1 = 0;  // owned routed experts [e0, e1) (SmallEP); the whole layer on one GPU
  int kbH = 0, kbI = 0, xs_stride = 0, hs_stride = 0;
  int rows_max = 0, tiles_max = 0, n_chunks_max = 0;
  int num_sms = 0;
  size_t slot_bytes = 0;
  int n_stage = 0;       // routed-expert slots currently in the pool (E when resident)
  int epl = 0;           // experts per launch (streamed)
  int residency = SLP_STREAMED;

  // resident device tensors
  uint16_t* d_router_hl = nullptr;  // [2][Erows][H] bf16 hi / lo split of router_w (tensor-core router)
  int Erows = 0;
  CUtensorMap tm_rw{};
  float *d_router_w = nullptr, *d_bias = nullptr, *d_gate_s = nullptr, *d_up_s = nullptr, *d_down_s = nullptr;
  uint8_t* d_pool = nullptr;  // [1 + n_stage] slots; slot 0 = shared expert
  // workspace
  float *d_logits = nullptr, *d_w = nullptr, *d_xs = nullptr, *d_hs = nullptr;
  int32_t *d_idx = nullptr, *d_counts = nullptr, *d_chunk = nullptr, *d_row_start = nullptr, *d_tile_start = nullptr,
          *d_tile_expert = nullptr, *d_pos = nullptr, *d_row_token = nullptr, *d_pair_start = nullptr, *d_pair_expert = nullptr;
  int4* d_tile_info = nullptr;
  uint8_t *d_xq = nullptr, *d_hq = nullptr;
  uint16_t* d_y = nullptr;  // [rows, H] fp16 per-row expert outputs, block-scaled by d_ys
  float* d_ys = nullptr;    // [rows, ys_stride] power-of-two scale per row per 128 columns
  int ys_stride = 0;
  int* d_err = nullptr;
  unsigned long long* d_clk = nullptr;
  int* d_sched = nullptr;
  void *d_e2e_in = nullptr, *d_e2e_out = nullptr;
  int32_t* h_counts = nullptr;  // pinned
  int* h_err = nullptr;         // pinned

  CUtensorMap tm_xq{}, tm_hq{}, tm_wgu{}, tm_wd{}, tm_y{};

  cudaStream_t copy_stream = nullptr, own_stream = nullptr;
  std::vector<cudaEvent_t> ev_ready, ev_free;
  std::vector<char> free_recorded;
  cudaEvent_t ev_done = nullptr, ev_t[6] = {}, ev_copy0 = nullptr, ev_copy1 = nullptr;
  int sh_rows = 0;  // rows of the shared expert's token range in the call being enqueued
  bool in_flight = false;
  bool dead = false;               // the expert pool could not be restored after a failed residency switch
  bool pool_needs_upload = false;  // resident pool was rebuilt after a failed switch: experts must be re-uploaded
  cudaStream_t last_stream = nullptr;
  int last_T = 0;
  slp_moe_stats stats{};
  bool stats_copy_valid = false;
  std::vector<cudaEvent_t> ev_k;  // 3 events per expert launch pair: before gate/up, between, after down
  std::vector<cudaEvent_t> ev_tail;  // ON events of the pieces of a call's last launch group
  struct Guarded { void* base; void* user; size_t bytes; const char* name; };
  std::vector<Guarded> guarded;      // triage "guards": workspace allocations with canary bands
  int ev_k_used = 0;
  int ev_k_shared = -1;  // first event of the shared expert's own launch pair in ev_k (-1: it shares a launch with routed experts)
};

namespace {

using L = slp_moe_layer;

// Workspace allocation.  With triage "guards" every buffer sits between two 4 KB canary bands (0xA5) that
// check_guards() reads back: a kernel that writes outside a buffer (the usual way a tile-bookkeeping bug shows) is
// caught without compute-sanitizer, which is closed on the GPU pool.
constexpr size_t kGuardBytes = 4096;
template <class T>
cudaError_t ws_alloc(L* h, T** out, size_t bytes, const char* name) {
  if (!h->triage.guards) return cudaMalloc(out, bytes);
  char* base = nullptr;
  const size_t padded = (bytes + 255) / 256 * 256;
  cudaError_t e = cudaMalloc(&base, padded + 2 * kGuardBytes);
  if (e != cudaSuccess) return e;
  e = cudaMemset(base, 0xA5, padded + 2 * kGuardBytes);
  if (e != cudaSuccess) return e;
  *out = reinterpret_cast<T*>(base + kGuardBytes);
  h->guarded.push_back({base, base + kGuardBytes, bytes, name});
  return cudaSuccess;
}
void ws_free(L* h, void* user) {
  if (!user) return;
  for (auto& gd : h->guarded)
    if (gd.user == user) { cudaFree(gd.base); gd.base = gd.user = nullptr; return; }
  cudaFree(user);
}
// Reads the canary bands back; the first damaged one is reported.
slp_status check_guards(L* h) {
  if (!h->triage.guards) return SLP_OK;
  std::vector<unsigned char> buf(kGuardBytes);
  for (const auto& gd : h->guarded) {
    if (!gd.base) continue;
    const size_t padded = (gd.bytes + 255) / 256 * 256;
    const char* bands[2] = {static_cast<const char*>(gd.base), static_cast<const char*>(gd.user) + padded};
    for (int b = 0; b < 2; ++b) {
      if (cudaMemcpy(buf.data(), bands[b], kGuardBytes, cudaMemcpyDeviceToHost) != cudaSuccess)
        return fail(SLP_ERR_CUDA, "reading the guard band of %s failed: %s", gd.name, cudaGetErrorString(cudaGetLastError()));
      for (size_t i = 0; i < kGuardBytes; ++i)
        if (buf[i] != 0xA5)
          return fail(SLP_ERR_CUDA, "guard band %s buffer %s (%zu bytes) overwritten at byte %zu", b ? "after" : "before", gd.name, gd.bytes, i);
    }
    // the slack between the buffer's end and the band (alignment padding) is canary too
    if (padded > gd.bytes) {
      const size_t n = padded - gd.bytes;
      if (cudaMemcpy(buf.data(), static_cast<const char*>(gd.user) + gd.bytes, n, cudaMemcpyDeviceToHost) != cudaSuccess)
        return fail(SLP_ERR_CUDA, "reading the slack of %s failed", gd.name);
      for (size_t i = 0; i < n; ++i)
        if (buf[i] != 0xA5) return fail(SLP_ERR_CUDA, "buffer %s (%zu bytes) overrun by %zu bytes", gd.name, gd.bytes, i + 1);
    }
  }
  return SLP_OK;
}

void select_layer(L* h, int l) {
  if (h->cur_layer == l) return;
  const LayerW& w = h->layers[l];
  h->hw = w.hw;
  h->gate_q = w.gate_q; h->up_q = w.up_q; h->down_q = w.down_q;
  h->d_router_hl = w.d_router_hl; h->tm_rw = w.tm_rw;
  h->d_router_w = w.d_router_w; h->d_bias = w.d_bias;
  h->d_gate_s = w.d_gate_s; h->d_up_s = w.d_up_s; h->d_down_s = w.d_down_s;
  h->d_shpool = w.d_shpool; h->tm_shgu = w.tm_shgu; h->tm_shd = w.tm_shd;
  h->cur_layer = l;
}
void stash_layer(L* h, int l) {  // the inverse, used while a layer's tensors are being created
  LayerW& w = h->layers[l];
  w.hw = h->hw;
  w.gate_q = h->gate_q; w.up_q = h->up_q; w.down_q = h->down_q;
  w.d_router_hl = h->d_router_hl; w.tm_rw = h->tm_rw;
  w.d_router_w = h->d_router_w; w.d_bias = h->d_bias;
  w.d_gate_s = h->d_gate_s; w.d_up_s = h->d_up_s; w.d_down_s = h->d_down_s;
  w.d_shpool = h->d_shpool; w.tm_shgu = h->tm_shgu; w.tm_shd = h->tm_shd;
}

struct Pool {
  uint8_t* d_pool = nullptr;
  std::vector<cudaEvent_t> ev_ready, ev_free;
  CUtensorMap tm_wgu{}, tm_wd{};
};

void release_pool(Pool* p) {
  if (p->d_pool) cudaFree(p->d_pool);
  p->d_pool = nullptr;
  for (auto e : p->ev_ready) cudaEventDestroy(e);
  for (auto e : p->ev_free) cudaEventDestroy(e);
  p->ev_ready.clear();
  p->ev_free.clear();
}

void free_pool(L* h) {
  Pool p;
  p.d_pool = h->d_pool;
  p.ev_ready.swap(h->ev_ready);
  p.ev_free.swap(h->ev_free);
  release_pool(&p);
  h->d_pool = nullptr;
  h->free_recorded.clear();
}

slp_status build_pool(L* h, int n_stage, int epl, Pool* p) {
  const size_t bytes = static_cast<size_t>(1 + n_stage) * h->slot_bytes;
  CU_TRY(cudaMalloc(&p->d_pool, bytes));
  const size_t IH = static_cast<size_t>(h->I) * h->H;
  // Pool layout: [gate of all slots | up of all slots | down of all slots], slot 0 = shared expert.
  // Kind-major so that experts that are contiguous in host memory (stacked [E, I, H] tensors, the usual
  // fused-MoE layout) land contiguously too and several experts travel in ONE cudaMemcpyAsync: the
  // ~4 us gap between back-to-back 14.7 MB copies is 1.5 % of the link time (profiles/r1_h2d_chunks.md).
  const size_t S = static_cast<size_t>(1 + n_stage);
  if (h->cfg.n_shared) {
    const slp_moe_host_weights& w0 = h->layers[0].hw;  // slot 0 = the shared expert of layer 0 (resident)
    CU_TRY(cudaMemcpy(p->d_pool, w0.shared_gate_q, IH, cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpy(p->d_pool + S * IH, w0.shared_up_q, IH, cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpy(p->d_pool + 2 * S * IH, w0.shared_down_q, IH, cudaMemcpyHostToDevice));
  } else {
    for (int kind = 0; kind < 3; ++kind) CU_TRY(cudaMemset(p->d_pool + kind * S * IH, 0, IH));
  }
  slp_status st = make_tmap_u8(&p->tm_wgu, p->d_pool, h->H, static_cast<uint64_t>(1 + n_stage) * 3 * h->I, slp::tc::kBoxRows);
  if (st != SLP_OK) return st;
  st = make_tmap_u8(&p->tm_wd, p->d_pool, h->I, static_cast<uint64_t>(1 + n_stage) * 3 * h->H, slp::tc::kBoxRows);
  if (st != SLP_OK) return st;
  const int n_groups = (n_stage + epl - 1) / epl;
  for (int i = 0; i < n_groups; ++i) {
    cudaEvent_t a = nullptr, b = nullptr;
    CU_TRY(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    p->ev_ready.push_back(a);
    CU_TRY(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    p->ev_free.push_back(b);
  }
  return SLP_OK;
}

// (Re)allocates the expert pool with `n_stage` routed slots (+ slot 0 for the shared expert), uploads
// the shared expert, rebuilds the weight tensor maps and the ring events.  `keep_old_until_built`:
// the new pool is built next to the old one and swapped in only on success, so a failure (out of
// memory on the way to resident mode) leaves the handle exactly as it was.  When both pools do not fit
// side by side the old one is released first; if the new one then fails, the previous pool is rebuilt,
// and only if that fails too is the handle marked dead (prefill then returns an error, never a launch
// against a null pool).
slp_status alloc_pool(L* h, int n_stage, int epl) {
  Pool fresh;
  slp_status st = build_pool(h, n_stage, epl, &fresh);
  if (st != SLP_OK && h->d_pool) {
    const std::string first_error = g_last_error;
    release_pool(&fresh);
    cudaGetLastError();
    const int old_stage = h->n_stage, old_epl = h->epl;
    free_pool(h);  // make room: the two pools did not fit side by side
    st = build_pool(h, n_stage, epl, &fresh);
    if (st != SLP_OK) {
      release_pool(&fresh);
      cudaGetLastError();
      Pool back;
      if (build_pool(h, old_stage, old_epl, &back) == SLP_OK) {
        h->d_pool = back.d_pool;
        h->ev_ready.swap(back.ev_ready);
        h->ev_free.swap(back.ev_free);
        h->tm_wgu = back.tm_wgu;
        h->tm_wd = back.tm_wd;
        h->free_recorded.assign(h->ev_ready.size(), 0);
        h->occ_layer.assign(h->ev_ready.size(), -1);
        h->occ_e0.assign(h->ev_ready.size(), -1);
        h->occ_prefetched.assign(h->ev_ready.size(), 0);
        h->pool_needs_upload = true;  // resident experts were lost with the old pool
      } else {
        release_pool(&back);
        cudaGetLastError();
        h->dead = true;
      }
      return fail(st, "expert pool of %d slots could not be allocated: %s", n_stage, first_error.c_str());
    }
  } else if (st != SLP_OK) {
    release_pool(&fresh);
    return st;
  }
  free_pool(h);
  h->d_pool = fresh.d_pool;
  h->ev_ready.swap(fresh.ev_ready);
  h->ev_free.swap(fresh.ev_free);
  h->tm_wgu = fresh.tm_wgu;
  h->tm_wd = fresh.tm_wd;
  h->free_recorded.assign(h->ev_ready.size(), 0);
  h->occ_layer.assign(h->ev_ready.size(), -1);
  h->occ_e0.assign(h->ev_ready.size(), -1);
  h->occ_prefetched.assign(h->ev_ready.size(), 0);
  h->n_stage = n_stage;
  h->epl = epl;
  return SLP_OK;
}

// Host ranges this library registered with cudaHostRegister, process wide, with a reference count: two handles may
// borrow the SAME host weight copy (prefill and decode share one resident DRAM copy, zero-copy), and
// the range must stay page-locked until the last of them is destroyed.
std::mutex g_reg_mutex;
struct Registered { int refs; size_t bytes; };
std::map<void*, Registered> g_registered;  // start of each range this library registered -> users, length

void unregister_host_range(void* p) {
  std::lock_guard<std::mutex> lock(g_reg_mutex);
  auto it = g_registered.find(p);
  if (it == g_registered.end()) return;
  if (--it->second.refs == 0) {
    cudaHostUnregister(p);
    g_registered.erase(it);
  }
}

// true if [p, p + bytes) is page-locked host memory as far as the runtime can tell (first and last byte)
bool range_is_pinned(const void* p, size_t bytes) {
  const char* ends[2] = {static_cast<const char*>(p), static_cast<const char*>(p) + (bytes ? bytes - 1 : 0)};
  for (const char* q : ends) {
    cudaPointerAttributes attr{};
    if (cudaPointerGetAttributes(&attr, q) != cudaSuccess || attr.type != cudaMemoryTypeHost) {
      cudaGetLastError();
      return false;
    }
  }
  return true;
}

slp_status pin_range(L* h, const void* p, size_t bytes, const char* what) {
  cudaPointerAttributes attr{};
  cudaError_t e = cudaPointerGetAttributes(&attr, p);
  if (e == cudaSuccess && attr.type == cudaMemoryTypeManaged)
    return fail(SLP_ERR_NOT_PINNED, "%s is managed memory: the streaming engine needs page-locked host memory "
                                    "(cudaMemcpyAsync from managed memory is staged and far below link rate)", what);
  if (e == cudaSuccess && attr.type == cudaMemoryTypeDevice)
    return fail(SLP_ERR_INVALID_ARG, "%s is a device pointer; host weights are expected", what);
  cudaGetLastError();
  // One lock over lookup, registration and insertion: two threads creating handles over the same host copy must not
  // both see "not registered yet", or one of them would hold the range without a reference and lose it at the
  // other's destroy.
  std::lock_guard<std::mutex> lock(g_reg_mutex);
  auto it = g_registered.find(const_cast<void*>(p));
  if (it != g_registered.end() && bytes <= it->second.bytes) {  // registered by another handle of this process: share it
    ++it->second.refs;
    h->registered.push_back(const_cast<void*>(p));
    return SLP_OK;
  }
  // (a range that starts at a registered pointer but is LONGER than what was registered, e.g. the full expert stack
  // after a shard of it, is not covered by that entry: it goes through the checks below like any other range)
  if (range_is_pinned(p, bytes)) return SLP_OK;
  if (h->cfg.require_pinned) return fail(SLP_ERR_NOT_PINNED, "%s is pageable host memory and require_pinned is set", what);
  e = cudaHostRegister(const_cast<void*>(p), bytes, cudaHostRegisterDefault);
  if (e == cudaErrorHostMemoryAlreadyRegistered) {
    // part of the range (a page shared with a neighbouring tensor, or a shorter range another handle registered) was
    // registered before: accept only if the whole range is page-locked now, otherwise the copies would silently fall
    // back to staged transfers
    cudaGetLastError();
    if (range_is_pinned(p, bytes)) return SLP_OK;
    return fail(SLP_ERR_NOT_PINNED, "%s overlaps an already registered range but is not page-locked end to end; "
                                    "register the enclosing allocation once or pass pinned memory", what);
  }
  if (e != cudaSuccess) return fail(SLP_ERR_NOT_PINNED, "cudaHostRegister(%s, %zu bytes) failed: %s", what, bytes, cudaGetErrorString(e));
  g_registered[const_cast<void*>(p)] = Registered{1, bytes};
  h->registered.push_back(const_cast<void*>(p));
  return SLP_OK;
}

slp_status wait_idle(L* h) {
  if (h->in_flight) {
    CU_TRY(cudaEventSynchronize(h->ev_done));
    h->in_flight = false;
  }
  return SLP_OK;
}

slp_status check_kernel_error(L* h) {
  if (*h->h_err != 0) {
    int code = *h->h_err;
    *h->h_err = 0;
    cudaMemset(h->d_err, 0, sizeof(int));
    return fail(SLP_ERR_KERNEL_TIMEOUT, "grouped GEMM pipeline wait timed out (role code %d)", code);
  }
  return SLP_OK;
}

slp::GemmArgs gemm_args(L* h, int mode, int e_begin, int e_end, int T) {
  slp::GemmArgs g{};
  const bool sh_own_pool = e_begin == h->E && h->d_shpool != nullptr;  // shared expert of a layer > 0
  g.tile_expert = h->d_tile_expert;
  g.tile_start = h->d_tile_start;
  g.row_start = h->d_row_start;
  g.counts = h->d_counts;
  g.tile_info = h->d_tile_info;
  g.pair_start = h->d_pair_start;
  g.pair_expert = h->d_pair_expert;
  g.e_begin = e_begin;
  g.e_end = e_end;
  g.E = h->E;
  g.T = T;
  g.e_own0 = h->e0;
  g.shared_rows = h->sh_rows;
  g.n_stage = h->n_stage;
  g.n_slots = sh_own_pool ? 1 : 1 + h->n_stage;
  g.a_q = mode == 0 ? h->d_xq : h->d_hq;
  g.a_s = mode == 0 ? h->d_xs : h->d_hs;
  g.a_s_stride = mode == 0 ? h->xs_stride : h->hs_stride;
  g.pool = sh_own_pool ? h->d_shpool : h->d_pool;
  g.gate_s = h->d_gate_s;
  g.up_s = h->d_up_s;
  g.down_s = h->d_down_s;
  g.H = h->H;
  g.I = h->I;
  g.hq = h->d_hq;
  g.hs = h->d_hs;
  g.hs_stride = h->hs_stride;
  g.y = h->d_y;
  g.ys = h->d_ys;
  g.ys_stride = h->ys_stride;
  g.err = h->d_err;
  g.clk = h->d_clk;
  g.sched = h->d_sched;
  return g;
}

// Launches gate/up (+SwiGLU+requant) and down for experts [e_begin, e_end) on `s`.
// `max_tiles` bounds the number of 128-row tiles in the range (host-side, no sync).
slp_status launch_experts(L* h, cudaStream_t s, int e_begin, int e_end, int T, int max_tiles) {
  if (h->triage.gemm == kGemmSimt) {
    slp::GemmArgs g0 = gemm_args(h, 0, e_begin, e_end, T), g1 = gemm_args(h, 1, e_begin, e_end, T);
    dim3 grid0(h->I / 128, max_tiles * 4), grid1(h->H / 128, max_tiles * 4);
    slp::gemm_simt_kernel<0><<<grid0, 256, 0, s>>>(g0);
    slp::gemm_simt_kernel<1><<<grid1, 256, 0, s>>>(g1);
  } else {
    slp::GemmArgs g0 = gemm_args(h, 0, e_begin, e_end, T), g1 = gemm_args(h, 1, e_begin, e_end, T);
    const int nt0 = h->I / 128, nt1 = (h->H + 255) / 256;
    const bool sh_own_pool = e_begin == h->E && h->d_shpool != nullptr;  // shared expert of a layer > 0: its own small pool
    const CUtensorMap& tm_wgu = sh_own_pool ? h->tm_shgu : h->tm_wgu;
    const CUtensorMap& tm_wd = sh_own_pool ? h->tm_shd : h->tm_wd;
    cudaEvent_t* ev = (h->ev_k_used + 3 <= static_cast<int>(h->ev_k.size())) ? &h->ev_k[h->ev_k_used] : nullptr;
    if (h->triage.gemm == kGemmTc) CU_TRY(cudaMemsetAsync(h->d_sched, 0, 2 * sizeof(int), s));  // work-item counters of the two launches below
    if (ev) cudaEventRecord(ev[0], s);
    if (h->triage.gemm == kGemmPair) {
      // CTA-pair kernel: clusters of two CTAs, one per SM; a work item is a pair of 128-row tiles
      namespace tc = slp::tc;
      const int n_cl = h->num_sms / 2;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeClusterDimension;
      attr[0].val.clusterDim.x = 2;
      attr[0].val.clusterDim.y = 1;
      attr[0].val.clusterDim.z = 1;
      cudaLaunchConfig_t lc{};
      lc.blockDim = dim3(tc::kThreads);
      lc.dynamicSmemBytes = tc::Cfg<0, true>::kSmemBytes;
      lc.stream = s;
      lc.attrs = attr;
      lc.numAttrs = 1;
      lc.gridDim = dim3(2 * std::max(1, std::min(n_cl, max_tiles * nt0)));
      CU_TRY(cudaLaunchKernelEx(&lc, tc::gemm_tc_kernel<0, true>, h->tm_xq, tm_wgu, h->tm_y, g0));
      if (ev) cudaEventRecord(ev[1], s);
      lc.gridDim = dim3(2 * std::max(1, std::min(n_cl, max_tiles * nt1)));
      lc.dynamicSmemBytes = tc::Cfg<1, true>::kSmemBytes;
      CU_TRY(cudaLaunchKernelEx(&lc, tc::gemm_tc_kernel<1, true>, h->tm_hq, tm_wd, h->tm_y, g1));
    } else {
      const int grid0 = std::max(1, std::min(h->num_sms, max_tiles * nt0));
      const int grid1 = std::max(1, std::min(h->num_sms, max_tiles * nt1));
      namespace tc = slp::tc;
      if (h->triage.gemm == kGemmTc) {  // dynamic tile distribution (the product path); 3 = static round-robin
        tc::gemm_tc_kernel<0, false, true><<<grid0, tc::kThreads, tc::Cfg<0, false>::kSmemBytes, s>>>(h->tm_xq, tm_wgu, h->tm_y, g0);
        if (ev) cudaEventRecord(ev[1], s);
        tc::gemm_tc_kernel<1, false, true><<<grid1, tc::kThreads, tc::Cfg<1, false>::kSmemBytes, s>>>(h->tm_hq, tm_wd, h->tm_y, g1);
      } else {
        tc::gemm_tc_kernel<0, false><<<grid0, tc::kThreads, tc::Cfg<0, false>::kSmemBytes, s>>>(h->tm_xq, tm_wgu, h->tm_y, g0);
        if (ev) cudaEventRecord(ev[1], s);
        tc::gemm_tc_kernel<1, false><<<grid1, tc::kThreads, tc::Cfg<1, false>::kSmemBytes, s>>>(h->tm_hq, tm_wd, h->tm_y, g1);
      }
    }
    if (ev) {
      cudaEventRecord(ev[2], s);
      if (e_begin == h->E) h->ev_k_shared = h->ev_k_used;  // the shared expert alone
      h->ev_k_used += 3;
    }
  }
  CU_TRY(cudaGetLastError());
  h->stats.gemm_launches += 2;
  h->stats.kernel_launches += 2;
  return SLP_OK;
}

// Enqueues the host -> HBM copies of the wanted experts of [e0, e1) on the copy stream.  Runs of
// experts whose host matrices AND ring slots are both consecutive are merged into one copy per kind.
slp_status copy_experts(L* h, int e0, int e1, const int32_t* counts /* NULL = all wanted */) {
  const size_t IH = static_cast<size_t>(h->I) * h->H, S = static_cast<size_t>(1 + h->n_stage);
  const std::vector<const uint8_t*>* src[3] = {&h->gate_q, &h->up_q, &h->down_q};
  auto wanted = [&](int e) { return !counts || counts[e] > 0; };
  for (int kind = 0; kind < 3; ++kind) {
    const std::vector<const uint8_t*>& p = *src[kind];
    uint8_t* region = h->d_pool + static_cast<size_t>(kind) * S * IH;
    for (int e = e0; e < e1;) {
      if (!wanted(e)) { ++e; continue; }
      int n = 1;  // experts e .. e + n - 1 in one copy
      while (e + n < e1 && wanted(e + n) && p[e + n] == p[e] + static_cast<size_t>(n) * IH &&
             (e + n - h->e0) % h->n_stage == (e - h->e0) % h->n_stage + n)
        ++n;
      CU_TRY(cudaMemcpyAsync(region + static_cast<size_t>(1 + (e - h->e0) % h->n_stage) * IH, p[e], static_cast<size_t>(n) * IH,
                             cudaMemcpyHostToDevice, h->copy_stream));
      h->stats.h2d_copies += 1;
      e += n;
    }
  }
  for (int e = e0; e < e1; ++e)
    if (wanted(e)) {
      h->stats.bytes_copied += static_cast<int64_t>(3 * IH);
      h->stats.experts_copied += 1;
    }
  return SLP_OK;
}

// `partial`: out is fp32 [T, H], the unrounded weighted sum over the owned experts (+ the shared expert for tokens
// in [sh_t0, sh_t1)); otherwise out is bf16 [T, H] and the shared expert covers every token.
slp_status prefetch_layer(L* h, int l);

slp_status prefill_impl(L* h, const void* hidden, int T, void* out, cudaStream_t s, bool partial = false, int sh_t0 = 0, int sh_t1 = -1,
                        int layer = 0) {
  const int E = h->E, k = h->k, H = h->H;
  select_layer(h, layer);
  if (sh_t1 < 0) sh_t1 = T;
  if (h->cfg.n_shared == 0) sh_t0 = sh_t1 = 0;
  const bool shared = sh_t1 > sh_t0;
  // The GEMMs run the shared expert over rows [sh_g0, sh_t1), sh_g0 = sh_t0 rounded down to a multiple of 32: the down
  // kernel stores Y / ys in whole 32-row groups counted from the range's first row, so a range that starts on a group
  // boundary ends its last group at roundup32(sh_t1) <= Tpad and cannot spill into the first routed expert's rows
  // (an arbitrary start could, by up to 31 rows, when sh_t1 is within 31 rows of Tpad).  The up to 31 extra rows in
  // front hold other tokens' quantised hidden states (quant_scatter writes every token's own row), their Y rows are
  // computed and never read: the combine kernel keeps the caller's [sh_t0, sh_t1).
  const int sh_g0 = shared ? (sh_t0 & ~31) : sh_t0;
  h->sh_rows = sh_t1 - sh_g0;
  const int e_own0 = h->e0, e_own1 = h->e1;
  h->stats = slp_moe_stats{};
  h->stats.struct_size = sizeof(slp_moe_stats);
  h->stats.tokens = T;
  h->stats.residency = h->residency;
  h->stats.layer = layer;
  h->stats_copy_valid = false;
  h->ev_k_used = 0;
  h->ev_k_shared = -1;
  auto launched = [&](int n) { h->stats.kernel_launches += n; };

  CU_TRY(cudaMemsetAsync(h->d_clk, 0, 16 * sizeof(unsigned long long), s));
  CU_TRY(cudaEventRecord(h->ev_t[0], s));
  // ---- a1 router ----
  {
    if (h->triage.router_fp32) {
      dim3 grid((T + 63) / 64, (E + 63) / 64);
      slp::router_logits_kernel<<<grid, 256, 0, s>>>(static_cast<const uint16_t*>(hidden), h->d_router_w, h->d_logits, T, H, E);
    } else {
      CUtensorMap tm_x;
      slp_status st = make_tmap_u8(&tm_x, const_cast<void*>(hidden), static_cast<uint64_t>(H) * 2, static_cast<uint64_t>(T));
      if (st != SLP_OK) return st;
      namespace rtc = slp::rtc;
      const int row_tiles = (T + rtc::BM - 1) / rtc::BM, n_tiles = (E + rtc::BN - 1) / rtc::BN;
      if (row_tiles * n_tiles > h->num_sms) {  // more than one wave of 128-token CTAs: two row tiles per CTA halve the W_r traffic
        dim3 grid((row_tiles + 1) / 2, n_tiles);
        rtc::router_logits_tc_kernel<2><<<grid, rtc::kThreads, rtc::Cfg<2>::kSmemBytes, s>>>(tm_x, h->tm_rw, h->d_logits, T, H, E, h->Erows, h->d_err);
      } else {
        dim3 grid(row_tiles, n_tiles);
        rtc::router_logits_tc_kernel<1><<<grid, rtc::kThreads, rtc::Cfg<1>::kSmemBytes, s>>>(tm_x, h->tm_rw, h->d_logits, T, H, E, h->Erows, h->d_err);
      }
    }
    const int warps = 8;
    const int blocks = (T + warps - 1) / warps;
    const float* bias = h->cfg.scoring == SLP_SCORE_SIGMOID_BIAS ? h->d_bias : nullptr;
    const int G = h->cfg.n_group;
    const bool fast = E % 32 == 0 && (E / 32 == 1 || E / 32 == 2 || E / 32 == 4 || E / 32 == 8 || E / 32 == 16) &&
                      (G & (G - 1)) == 0 && G <= 32;
#define SLP_TOPK_FAST(P)                                                                                              \
  slp::router_topk_fast_kernel<P><<<blocks, warps * 32, 0, s>>>(h->d_logits, bias, h->d_idx, h->d_w, T, k, G,         \
                                                                h->cfg.topk_group, h->cfg.scoring, h->cfg.norm_topk, \
                                                                h->cfg.routed_scale)
    if (fast) {  // contiguous experts per lane: groups are runs of lanes (kernels_route.cuh)
      switch (E / 32) {
        case 1: SLP_TOPK_FAST(1); break;
        case 2: SLP_TOPK_FAST(2); break;
        case 4: SLP_TOPK_FAST(4); break;
        case 8: SLP_TOPK_FAST(8); break;
        default: SLP_TOPK_FAST(16); break;
      }
    } else
#undef SLP_TOPK_FAST
    if (E <= 128)
      slp::router_topk_kernel<4><<<blocks, warps * 32, 0, s>>>(h->d_logits, bias, h->d_idx, h->d_w, T, E, k, h->cfg.n_group,
                                                               h->cfg.topk_group, h->cfg.scoring, h->cfg.norm_topk, h->cfg.routed_scale);
    else if (E <= 256)
      slp::router_topk_kernel<8><<<blocks, warps * 32, 0, s>>>(h->d_logits, bias, h->d_idx, h->d_w, T, E, k, h->cfg.n_group,
                                                               h->cfg.topk_group, h->cfg.scoring, h->cfg.norm_topk, h->cfg.routed_scale);
    else
      slp::router_topk_kernel<16><<<blocks, warps * 32, 0, s>>>(h->d_logits, bias, h->d_idx, h->d_w, T, E, k, h->cfg.n_group,
                                                                h->cfg.topk_group, h->cfg.scoring, h->cfg.norm_topk, h->cfg.routed_scale);
    launched(2);
  }
  // ---- a2 histogram / scan / permute ----
  const int n_chunks = (T + slp::kChunkTokens - 1) / slp::kChunkTokens;
  {
    const int wpb = 4;
    const int blocks = (n_chunks + wpb - 1) / wpb;
    const size_t sm = static_cast<size_t>(wpb) * E * sizeof(int32_t);
    CU_TRY(cudaMemsetAsync(h->d_row_token, 0xFF, static_cast<size_t>(h->rows_max) * sizeof(int32_t), s));
    slp::permute_hist_kernel<<<blocks, wpb * 32, sm, s>>>(h->d_idx, h->d_chunk, T, k, E);
    slp::permute_scan_kernel<<<1, 512, 0, s>>>(h->d_chunk, h->d_counts, h->d_row_start, h->d_tile_start, h->d_tile_expert, h->d_pair_start, h->d_pair_expert, h->d_tile_info, n_chunks, T,
                                               E, e_own0, e_own1, sh_g0, sh_t1);
    slp::permute_place_kernel<<<blocks, wpb * 32, sm, s>>>(h->d_idx, h->d_chunk, h->d_row_start, h->d_pos, h->d_row_token, T, k, E, e_own0, e_own1);
    launched(3);
  }
  // ---- a3 hidden quantisation + scatter into expert order ----
  slp::quant_scatter_kernel<<<T, 256, 0, s>>>(static_cast<const uint16_t*>(hidden), h->d_pos, h->d_xq, h->d_xs, T, H, k, h->xs_stride);
  launched(1);
  CU_TRY(cudaGetLastError());
  CU_TRY(cudaEventRecord(h->ev_t[1], s));

  const int Tpad_tiles = (h->sh_rows + 127) / 128;
  const int routed_tiles_bound = (T * k) / 128 + (e_own1 - e_own0);
  h->stats.m_tiles = 0;

  bool skip = h->cfg.skip_empty_experts != 0;
  if (skip) {
    CU_TRY(cudaMemcpyAsync(h->h_counts, h->d_counts, E * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    CU_TRY(cudaStreamSynchronize(s));
  }

  CU_TRY(cudaEventRecord(h->ev_t[2], s));
  if (h->residency == SLP_RESIDENT) {
    // one launch pair covers the owned routed experts and, when it is adjacent (e_own1 == E), the shared expert
    if (e_own1 == E || !shared) {
      slp_status st = launch_experts(h, s, e_own0, shared ? E + 1 : e_own1, T, routed_tiles_bound + (shared ? Tpad_tiles : 0));
      if (st != SLP_OK) return st;
    } else {
      slp_status st = launch_experts(h, s, e_own0, e_own1, T, routed_tiles_bound);
      if (st != SLP_OK) return st;
      st = launch_experts(h, s, E, E + 1, T, Tpad_tiles);
      if (st != SLP_OK) return st;
    }
  } else {
    // ---- a4 streaming engine ----
    if (shared) {  // resident weights: runs while the first expert copies are in flight
      slp_status st = launch_experts(h, s, E, E + 1, T, Tpad_tiles);
      if (st != SLP_OK) return st;
    }
    const int epl = h->epl;
    const int n_ring = static_cast<int>(h->ev_ready.size());
    bool first_copy = true;
    for (int e0 = e_own0, grp = 0; e0 < e_own1; e0 += epl, ++grp) {
      const int e1 = std::min(e_own1, e0 + epl);
      const int r = grp % n_ring;
      int need = 0, rows_bound = 0;
      for (int e = e0; e < e1; ++e) {
        const bool want = !skip || h->h_counts[e] > 0;
        need += want ? 1 : 0;
        if (skip) rows_bound += (h->h_counts[e] + 127) / 128;
      }
      if (need == 0) {
        h->stats.experts_skipped += e1 - e0;
        if (h->occ_prefetched[r] && h->occ_layer[r] == layer && h->occ_e0[r] == e0) h->occ_prefetched[r] = 0;  // loaded ahead, not needed after all
        continue;
      }
      // already loaded (or loading) by an earlier call's run-ahead?  then this call only waits for its ON event
      const bool have = h->occ_prefetched[r] && h->occ_layer[r] == layer && h->occ_e0[r] == e0;
      if (have) {
        h->stats.experts_from_prefetch += e1 - e0;
      } else {
        if (h->free_recorded[r]) CU_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_free[r], 0));  // OFF -> slot reusable
        if (first_copy) {
          CU_TRY(cudaEventRecord(h->ev_copy0, h->copy_stream));
          first_copy = false;
        }
        for (int e = e0; e < e1; ++e)
          if (skip && h->h_counts[e] == 0) h->stats.experts_skipped += 1;
        // The call ends one group's compute after the last copy has landed.  The LAST group of a long call is therefore
        // copied and launched in pieces of kTailExperts experts, each launch waiting only for its own piece: the tail
        // shrinks from the compute of a whole group (3.3 ms of a 32K-token call with 64 experts per launch) to that
        // of a piece, while every other group keeps the large launches that amortise the launch ramp.
        // Only where it pays: with fewer than ~256 rows per expert the GEMMs are HBM-bound, the whole group's compute is
        // well under a millisecond and small launches would only add launch ramps.
        const bool last_group = e1 == e_own1 && e1 - e0 > kTailExperts && !h->ev_tail.empty() &&
                                static_cast<long long>(T) * k >= 256LL * E;
        if (last_group) {
          int piece = 0;
          for (int p0 = e0; p0 < e1; p0 += kTailExperts, ++piece) {
            const int p1 = std::min(e1, p0 + kTailExperts);
            int pneed = 0, prows = 0;
            for (int e = p0; e < p1; ++e) {
              pneed += (!skip || h->h_counts[e] > 0) ? 1 : 0;
              if (skip) prows += (h->h_counts[e] + 127) / 128;
            }
            if (pneed == 0) continue;
            slp_status st = copy_experts(h, p0, p1, skip ? h->h_counts : nullptr);
            if (st != SLP_OK) return st;
            cudaEvent_t ev = h->ev_tail[piece % h->ev_tail.size()];
            CU_TRY(cudaEventRecord(ev, h->copy_stream));
            CU_TRY(cudaStreamWaitEvent(s, ev, 0));
            const int pbound = skip ? prows : std::min(routed_tiles_bound, (T * k) / 128 + (p1 - p0));
            st = launch_experts(h, s, p0, p1, T, std::max(1, pbound));
            if (st != SLP_OK) return st;
          }
          h->occ_layer[r] = layer;
          h->occ_e0[r] = e0;
          h->occ_prefetched[r] = 0;
          CU_TRY(cudaEventRecord(h->ev_ready[r], h->copy_stream));  // ON for the whole group (bookkeeping of later calls)
          CU_TRY(cudaEventRecord(h->ev_free[r], s));  // OFF
          h->free_recorded[r] = 1;
          continue;
        }
        {
          slp_status st = copy_experts(h, e0, e1, skip ? h->h_counts : nullptr);
          if (st != SLP_OK) return st;
        }
        CU_TRY(cudaEventRecord(h->ev_ready[r], h->copy_stream));  // ON
        h->occ_layer[r] = layer;
        h->occ_e0[r] = e0;
      }
      h->occ_prefetched[r] = 0;
      CU_TRY(cudaStreamWaitEvent(s, h->ev_ready[r], 0));
      const int bound = skip ? rows_bound : std::min(routed_tiles_bound, (T * k) / 128 + (e1 - e0));
      slp_status st = launch_experts(h, s, e0, e1, T, std::max(1, bound));
      if (st != SLP_OK) return st;
      CU_TRY(cudaEventRecord(h->ev_free[r], s));  // OFF
      h->free_recorded[r] = 1;
    }
    // the loader keeps going with the next layer's modules (Fig. 5)
    const int n_layers = static_cast<int>(h->layers.size());
    if (n_layers > 1) {
      const int64_t b0 = h->stats.bytes_copied;
      const int32_t c0 = h->stats.experts_copied;
      if (first_copy) {
        CU_TRY(cudaEventRecord(h->ev_copy0, h->copy_stream));
        first_copy = false;
      }
      slp_status st = prefetch_layer(h, (layer + 1) % n_layers);
      if (st != SLP_OK) return st;
      h->stats.bytes_prefetched = h->stats.bytes_copied - b0;   // accounted apart from this layer's own weight pass
      h->stats.experts_prefetched = h->stats.experts_copied - c0;
      h->stats.bytes_copied = b0;
      h->stats.experts_copied = c0;
      select_layer(h, layer);
    }
    if (!first_copy) {
      CU_TRY(cudaEventRecord(h->ev_copy1, h->copy_stream));
      h->stats_copy_valid = true;
    }
  }
  CU_TRY(cudaEventRecord(h->ev_t[3], s));
  // ---- a9 combine ----
  if (partial) slp::combine_kernel<true><<<T, 256, 0, s>>>(h->d_y, h->d_ys, h->d_pos, h->d_w, out, T, H, k, sh_t0, sh_t1, h->ys_stride);
  else slp::combine_kernel<false><<<T, 256, 0, s>>>(h->d_y, h->d_ys, h->d_pos, h->d_w, out, T, H, k, sh_t0, sh_t1, h->ys_stride);
  launched(1);
  CU_TRY(cudaGetLastError());
  CU_TRY(cudaMemcpyAsync(h->h_err, h->d_err, sizeof(int), cudaMemcpyDeviceToHost, s));
  CU_TRY(cudaEventRecord(h->ev_t[4], s));
  CU_TRY(cudaEventRecord(h->ev_done, s));
  h->in_flight = true;
  h->last_stream = s;
  h->last_T = T;
  return SLP_OK;
}

// Loader run-ahead: enqueue the copies of layer l's launch groups into the ring (one pass over the ring at most);
// slots that already hold an unconsumed prefetch of the same group are kept, unconsumed prefetches of anything else are
// overwritten.  Each copy waits for the OFF event of the
// launch that last used its slot.  Leaves layer l selected.
slp_status prefetch_layer(L* h, int l) {
  if (h->residency != SLP_STREAMED) return SLP_OK;
  select_layer(h, l);
  const int epl = h->epl, n_ring = static_cast<int>(h->ev_ready.size());
  int grp = 0;
  for (int e0 = h->e0; e0 < h->e1 && grp < n_ring; e0 += epl, ++grp) {
    const int e1 = std::min(h->e1, e0 + epl), r = grp % n_ring;
    if (h->occ_prefetched[r]) {
      if (h->occ_layer[r] == l && h->occ_e0[r] == e0) continue;  // this very group is already loaded (or loading)
      // A prefetch for another layer or group that no call consumed (layers called out of order; its group turned out
      // empty under skip_empty_experts): it would otherwise sit there for ever and stop every later run-ahead at this
      // slot.  Overwrite it: the copy stream is in order, so the new copy follows the stale one, and the wait below
      // covers the last launch that read the slot.
    }
    if (h->free_recorded[r]) CU_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_free[r], 0));
    slp_status st = copy_experts(h, e0, e1, nullptr);
    if (st != SLP_OK) return st;
    CU_TRY(cudaEventRecord(h->ev_ready[r], h->copy_stream));
    h->occ_layer[r] = l;
    h->occ_e0[r] = e0;
    h->occ_prefetched[r] = 1;
  }
  return SLP_OK;
}

}  // namespace

extern "C" {

const char* slp_last_error(void) { return g_last_error.c_str(); }

slp_status slp_moe_debug_set_triage(const char* spec) {
  Triage t;
  std::string bad;
  if (spec && !parse_triage(spec, &t, &bad)) return fail(SLP_ERR_INVALID_ARG, "unknown triage token '%s'", bad.c_str());
  g_triage_next = t;
  return SLP_OK;
}
const char* slp_version(void) { return "slpmoe 0.3 (sm_100a; abi 3)"; }


slp_status slp_moe_layer_create(const slp_moe_cfg* cfg, const slp_moe_host_weights* w, slp_moe_layer** out) {
  return slp_moe_stack_create(cfg, 1, w, out);
}

slp_status slp_moe_stack_create(const slp_moe_cfg* cfg, int32_t n_layers, const slp_moe_host_weights* w_all, slp_moe_layer** out) {
  if (!cfg || !w_all || !out) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  if (n_layers < 1 || n_layers > 4096) return fail(SLP_ERR_INVALID_ARG, "n_layers %d outside 1..4096", n_layers);
  const slp_moe_host_weights* w = w_all;
  if (cfg->struct_size != sizeof(slp_moe_cfg))
    return fail(SLP_ERR_INVALID_ARG, "cfg.struct_size %u != %zu: the caller was built against another slp_moe.h (this library: ABI %u)",
                cfg->struct_size, sizeof(slp_moe_cfg), SLP_MOE_ABI_VERSION);
  if (cfg->abi_version != SLP_MOE_ABI_VERSION)
    return fail(SLP_ERR_INVALID_ARG, "cfg.abi_version %u, this library implements ABI %u", cfg->abi_version, SLP_MOE_ABI_VERSION);
  *out = nullptr;
  const int H = cfg->hidden, E = cfg->n_experts, k = cfg->top_k, I = cfg->moe_intermediate;
  int n_stage = 0, epl = 0;
  {
    slp_status vst = validate_cfg(cfg, &n_stage, &epl);
    if (vst != SLP_OK) return vst;
  }
  for (int l = 0; l < n_layers; ++l) {
    const slp_moe_host_weights* wl = w_all + l;
    if (!wl->router_w || !wl->gate_q || !wl->gate_s || !wl->up_q || !wl->up_s || !wl->down_q || !wl->down_s)
      return fail(SLP_ERR_INVALID_ARG, "NULL weight pointer (layer %d)", l);
    if (cfg->n_shared && (!wl->shared_gate_q || !wl->shared_gate_s || !wl->shared_up_q || !wl->shared_up_s || !wl->shared_down_q || !wl->shared_down_s))
      return fail(SLP_ERR_INVALID_ARG, "n_shared == 1 but a shared weight pointer is NULL (layer %d)", l);
  }

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(SLP_ERR_CUDA, "no CUDA device available (this library has no CPU path)");
  }
  if (cfg->device < 0 || cfg->device >= ndev) return fail(SLP_ERR_INVALID_ARG, "device %d out of range", cfg->device);
  CU_TRY(cudaSetDevice(cfg->device));
  cudaDeviceProp prop{};
  CU_TRY(cudaGetDeviceProperties(&prop, cfg->device));
  if (prop.major != 10) return fail(SLP_ERR_CUDA, "device %d is sm_%d%d; this library is built for sm_100a only", cfg->device, prop.major, prop.minor);

  L* h = new (std::nothrow) L();
  if (!h) return fail(SLP_ERR_OOM, "out of host memory");
  h->cfg = *cfg;
  h->triage = read_triage();
  h->layers.resize(n_layers);
  h->H = H; h->E = E; h->k = k; h->I = I; h->Tm = cfg->max_tokens;
  h->e0 = cfg->expert_end == 0 ? 0 : cfg->expert_begin;
  h->e1 = cfg->expert_end == 0 ? E : cfg->expert_end;
  h->kbH = H / 128; h->kbI = I / 128;
  h->xs_stride = round_up(h->kbH, 4);
  h->hs_stride = round_up(h->kbI, 4);
  h->ys_stride = round_up(h->kbH, 4);
  h->num_sms = prop.multiProcessorCount;
  h->slot_bytes = static_cast<size_t>(3) * I * H;
  const int Tpad = round_up(h->Tm, 128);
  h->rows_max = Tpad + round_up(h->Tm * k + E * 127, 128);
  h->tiles_max = h->rows_max / 128 + 1;
  h->n_chunks_max = (h->Tm + slp::kChunkTokens - 1) / slp::kChunkTokens;
  auto bail = [&](slp_status st) {
    std::string keep = g_last_error;
    slp_moe_layer_destroy(h);
    g_last_error = keep;
    return st;
  };
#define TRY_OR_BAIL(expr)                         \
  do {                                            \
    slp_status _s = (expr);                       \
    if (_s != SLP_OK) return bail(_s);            \
  } while (0)
#define CU_OR_BAIL(expr)                                                                                        \
  do {                                                                                                          \
    cudaError_t _e = (expr);                                                                                    \
    if (_e != cudaSuccess)                                                                                      \
      return bail(fail(_e == cudaErrorMemoryAllocation ? SLP_ERR_OOM : SLP_ERR_CUDA, "%s failed: %s", #expr,    \
                       cudaGetErrorString(_e)));                                                                \
  } while (0)

  const size_t IH = static_cast<size_t>(I) * H;
  CU_OR_BAIL(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  CU_OR_BAIL(cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking));
  CU_OR_BAIL(cudaEventCreateWithFlags(&h->ev_done, cudaEventDisableTiming));
  for (auto& e : h->ev_t) CU_OR_BAIL(cudaEventCreate(&e));
  CU_OR_BAIL(cudaEventCreate(&h->ev_copy0));
  CU_OR_BAIL(cudaEventCreate(&h->ev_copy1));
  h->ev_k.resize(3 * (E + 2));
  for (auto& e : h->ev_k) CU_OR_BAIL(cudaEventCreate(&e));
  h->ev_tail.resize(64);
  for (auto& e : h->ev_tail) CU_OR_BAIL(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));

  // ---- per layer: pin (or check) the streamed weights, upload router / bias / block scales / shared expert ----
  CU_OR_BAIL(cudaFuncSetAttribute(slp::rtc::router_logits_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::rtc::Cfg<1>::kSmemBytes));
  CU_OR_BAIL(cudaFuncSetAttribute(slp::rtc::router_logits_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::rtc::Cfg<2>::kSmemBytes));
  for (int l = 0; l < n_layers; ++l) {
    w = w_all + l;
    h->hw = *w;
    h->gate_q.assign(w->gate_q, w->gate_q + E);
    h->up_q.assign(w->up_q, w->up_q + E);
    h->down_q.assign(w->down_q, w->down_q + E);
    h->d_router_hl = nullptr; h->d_router_w = h->d_bias = h->d_gate_s = h->d_up_s = h->d_down_s = nullptr; h->d_shpool = nullptr;
    h->cur_layer = l;
    // (a failure below goes through bail -> destroy, which first stashes this half-built layer so that its tensors are freed)
  for (int e = h->e0; e < h->e1; ++e)
    if (!h->gate_q[e] || !h->up_q[e] || !h->down_q[e] || !w->gate_s[e] || !w->up_s[e] || !w->down_s[e])
      return bail(fail(SLP_ERR_INVALID_ARG, "NULL weight pointer for expert %d", e));
  {
    // Experts stacked in one [E, I, H] host tensor are checked / registered as ONE range per run: adjacent
    // matrices of a pageable allocation share a page, which cudaHostRegister refuses matrix by matrix.
    const std::vector<const uint8_t*>* kinds[3] = {&h->gate_q, &h->up_q, &h->down_q};
    const char* names[3] = {"gate_q", "up_q", "down_q"};
    for (int kind = 0; kind < 3; ++kind) {
      const std::vector<const uint8_t*>& p = *kinds[kind];
      for (int e = h->e0; e < h->e1;) {
        int n = 1;
        while (e + n < h->e1 && p[e + n] == p[e] + static_cast<size_t>(n) * IH) ++n;
        TRY_OR_BAIL(pin_range(h, p[e], static_cast<size_t>(n) * IH, names[kind]));
        e += n;
      }
    }
  }

  // resident tensors: router, bias, all block scales (entry E = shared expert)
  const size_t sc_gu = static_cast<size_t>(h->kbI) * h->kbH, sc_d = static_cast<size_t>(h->kbH) * h->kbI;
  CU_OR_BAIL(cudaMalloc(&h->d_router_w, static_cast<size_t>(E) * H * sizeof(float)));
  CU_OR_BAIL(cudaMemcpy(h->d_router_w, w->router_w, static_cast<size_t>(E) * H * sizeof(float), cudaMemcpyHostToDevice));
  {  // bf16 hi / lo split of the router weights for the tensor-core logits kernel
    h->Erows = round_up(E, slp::rtc::BN);
    const size_t hl_bytes = static_cast<size_t>(2) * h->Erows * H * sizeof(uint16_t);
    CU_OR_BAIL(cudaMalloc(&h->d_router_hl, hl_bytes));
    CU_OR_BAIL(cudaMemset(h->d_router_hl, 0, hl_bytes));
    slp::rtc::split_router_w_kernel<<<h->num_sms * 4, 256>>>(h->d_router_w, h->d_router_hl, E, H, h->Erows);
    CU_OR_BAIL(cudaGetLastError());
    TRY_OR_BAIL(make_tmap_u8(&h->tm_rw, h->d_router_hl, static_cast<uint64_t>(H) * 2, static_cast<uint64_t>(2) * h->Erows));
  }
  CU_OR_BAIL(cudaMalloc(&h->d_bias, E * sizeof(float)));
  if (w->router_bias) CU_OR_BAIL(cudaMemcpy(h->d_bias, w->router_bias, E * sizeof(float), cudaMemcpyHostToDevice));
  else CU_OR_BAIL(cudaMemset(h->d_bias, 0, E * sizeof(float)));
  CU_OR_BAIL(cudaMalloc(&h->d_gate_s, (E + 1) * sc_gu * sizeof(float)));
  CU_OR_BAIL(cudaMalloc(&h->d_up_s, (E + 1) * sc_gu * sizeof(float)));
  CU_OR_BAIL(cudaMalloc(&h->d_down_s, (E + 1) * sc_d * sizeof(float)));
  for (int e = h->e0; e < h->e1; ++e) {
    CU_OR_BAIL(cudaMemcpy(h->d_gate_s + e * sc_gu, w->gate_s[e], sc_gu * sizeof(float), cudaMemcpyHostToDevice));
    CU_OR_BAIL(cudaMemcpy(h->d_up_s + e * sc_gu, w->up_s[e], sc_gu * sizeof(float), cudaMemcpyHostToDevice));
    CU_OR_BAIL(cudaMemcpy(h->d_down_s + e * sc_d, w->down_s[e], sc_d * sizeof(float), cudaMemcpyHostToDevice));
  }
  if (cfg->n_shared) {
    CU_OR_BAIL(cudaMemcpy(h->d_gate_s + E * sc_gu, w->shared_gate_s, sc_gu * sizeof(float), cudaMemcpyHostToDevice));
    CU_OR_BAIL(cudaMemcpy(h->d_up_s + E * sc_gu, w->shared_up_s, sc_gu * sizeof(float), cudaMemcpyHostToDevice));
    CU_OR_BAIL(cudaMemcpy(h->d_down_s + E * sc_d, w->shared_down_s, sc_d * sizeof(float), cudaMemcpyHostToDevice));
  }

    if (cfg->n_shared && l > 0) {  // layer 0's shared expert lives in slot 0 of the ring pool
      CU_OR_BAIL(cudaMalloc(&h->d_shpool, 3 * IH));
      CU_OR_BAIL(cudaMemcpy(h->d_shpool, w->shared_gate_q, IH, cudaMemcpyHostToDevice));
      CU_OR_BAIL(cudaMemcpy(h->d_shpool + IH, w->shared_up_q, IH, cudaMemcpyHostToDevice));
      CU_OR_BAIL(cudaMemcpy(h->d_shpool + 2 * IH, w->shared_down_q, IH, cudaMemcpyHostToDevice));
      TRY_OR_BAIL(make_tmap_u8(&h->tm_shgu, h->d_shpool, h->H, static_cast<uint64_t>(3) * h->I, slp::tc::kBoxRows));
      TRY_OR_BAIL(make_tmap_u8(&h->tm_shd, h->d_shpool, h->I, static_cast<uint64_t>(3) * h->H, slp::tc::kBoxRows));
    }
    stash_layer(h, l);
  }
  h->cur_layer = -1;
  select_layer(h, 0);

  // workspace
  const size_t Tm = h->Tm, rows = h->rows_max;
  CU_OR_BAIL(ws_alloc(h, &h->d_logits, Tm * E * sizeof(float), "d_logits"));
  CU_OR_BAIL(ws_alloc(h, &h->d_idx, Tm * k * sizeof(int32_t), "d_idx"));
  CU_OR_BAIL(ws_alloc(h, &h->d_w, Tm * k * sizeof(float), "d_w"));
  CU_OR_BAIL(ws_alloc(h, &h->d_counts, E * sizeof(int32_t), "d_counts"));
  CU_OR_BAIL(ws_alloc(h, &h->d_chunk, static_cast<size_t>(h->n_chunks_max) * E * sizeof(int32_t), "d_chunk"));
  CU_OR_BAIL(ws_alloc(h, &h->d_row_start, (E + 2) * sizeof(int32_t), "d_row_start"));
  CU_OR_BAIL(ws_alloc(h, &h->d_tile_start, (E + 2) * sizeof(int32_t), "d_tile_start"));
  CU_OR_BAIL(ws_alloc(h, &h->d_tile_expert, static_cast<size_t>(h->tiles_max) * sizeof(int32_t), "d_tile_expert"));
  CU_OR_BAIL(ws_alloc(h, &h->d_tile_info, static_cast<size_t>(h->tiles_max) * sizeof(int4), "d_tile_info"));
  CU_OR_BAIL(ws_alloc(h, &h->d_pair_start, (E + 2) * sizeof(int32_t), "d_pair_start"));
  CU_OR_BAIL(ws_alloc(h, &h->d_pair_expert, static_cast<size_t>(h->tiles_max) * sizeof(int32_t), "d_pair_expert"));
  CU_OR_BAIL(ws_alloc(h, &h->d_pos, Tm * k * sizeof(int32_t), "d_pos"));
  CU_OR_BAIL(ws_alloc(h, &h->d_row_token, rows * sizeof(int32_t), "d_row_token"));
  CU_OR_BAIL(ws_alloc(h, &h->d_xq, rows * H, "d_xq"));
  CU_OR_BAIL(ws_alloc(h, &h->d_xs, rows * h->xs_stride * sizeof(float), "d_xs"));
  CU_OR_BAIL(ws_alloc(h, &h->d_hq, rows * I, "d_hq"));
  CU_OR_BAIL(ws_alloc(h, &h->d_hs, rows * h->hs_stride * sizeof(float), "d_hs"));
  CU_OR_BAIL(ws_alloc(h, &h->d_y, rows * H * sizeof(uint16_t), "d_y"));
  CU_OR_BAIL(ws_alloc(h, &h->d_ys, rows * h->ys_stride * sizeof(float), "d_ys"));
  CU_OR_BAIL(ws_alloc(h, &h->d_clk, 16 * sizeof(unsigned long long), "d_clk"));
  CU_OR_BAIL(ws_alloc(h, &h->d_sched, 2 * sizeof(int), "d_sched"));
  CU_OR_BAIL(ws_alloc(h, &h->d_err, sizeof(int), "d_err"));
  if (h->triage.guards == 2) CU_OR_BAIL(cudaMemset(reinterpret_cast<char*>(h->d_counts + E), 0, 1));  // negative control of the canary check
  CU_OR_BAIL(cudaMemset(h->d_err, 0, sizeof(int)));
  CU_OR_BAIL(cudaMemset(h->d_tile_expert, 0, static_cast<size_t>(h->tiles_max) * sizeof(int32_t)));
  CU_OR_BAIL(cudaMemset(h->d_tile_info, 0, static_cast<size_t>(h->tiles_max) * sizeof(int4)));
  CU_OR_BAIL(cudaMemset(h->d_pair_expert, 0, static_cast<size_t>(h->tiles_max) * sizeof(int32_t)));
  // padding rows are read by the tensor cores (their outputs are discarded): keep them finite
  CU_OR_BAIL(cudaMemset(h->d_xq, 0, rows * H));
  CU_OR_BAIL(cudaMemset(h->d_hq, 0, rows * I));
  CU_OR_BAIL(cudaMallocHost(&h->h_counts, E * sizeof(int32_t)));
  CU_OR_BAIL(cudaMallocHost(&h->h_err, sizeof(int)));
  *h->h_err = 0;

  TRY_OR_BAIL(make_tmap_u8(&h->tm_xq, h->d_xq, H, rows));
  TRY_OR_BAIL(make_tmap_u8(&h->tm_hq, h->d_hq, I, rows));
  TRY_OR_BAIL(make_tmap_f16_store(&h->tm_y, h->d_y, H, rows));
  TRY_OR_BAIL(alloc_pool(h, n_stage, epl));

  CU_OR_BAIL(cudaFuncSetAttribute(slp::tc::gemm_tc_kernel<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::tc::Cfg<0, true>::kSmemBytes));
  CU_OR_BAIL(cudaFuncSetAttribute(slp::tc::gemm_tc_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::tc::Cfg<1, true>::kSmemBytes));
  CU_OR_BAIL(cudaFuncSetAttribute(slp::tc::gemm_tc_kernel<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::tc::Cfg<0, false>::kSmemBytes));
  CU_OR_BAIL(cudaFuncSetAttribute(slp::tc::gemm_tc_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::tc::Cfg<1, false>::kSmemBytes));
  CU_OR_BAIL(cudaFuncSetAttribute(slp::tc::gemm_tc_kernel<0, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::tc::Cfg<0, false>::kSmemBytes));
  CU_OR_BAIL(cudaFuncSetAttribute(slp::tc::gemm_tc_kernel<1, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slp::tc::Cfg<1, false>::kSmemBytes));
  CU_OR_BAIL(cudaDeviceSynchronize());
#undef TRY_OR_BAIL
#undef CU_OR_BAIL
  *out = h;
  return SLP_OK;
}

slp_status slp_moe_query_plan(const slp_moe_cfg* cfg, slp_moe_plan* plan) {
  if (!cfg || !plan) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  if (cfg->struct_size != sizeof(slp_moe_cfg))
    return fail(SLP_ERR_INVALID_ARG, "cfg.struct_size %u != %zu: the caller was built against another slp_moe.h (this library: ABI %u)",
                cfg->struct_size, sizeof(slp_moe_cfg), SLP_MOE_ABI_VERSION);
  if (cfg->abi_version != SLP_MOE_ABI_VERSION)
    return fail(SLP_ERR_INVALID_ARG, "cfg.abi_version %u, this library implements ABI %u", cfg->abi_version, SLP_MOE_ABI_VERSION);
  if (plan->struct_size != sizeof(slp_moe_plan)) return fail(SLP_ERR_INVALID_ARG, "plan.struct_size mismatch");
  int n_stage = 0, epl = 0;
  slp_status st = validate_cfg(cfg, &n_stage, &epl);
  if (st != SLP_OK) return st;
  const int64_t H = cfg->hidden, E = cfg->n_experts, k = cfg->top_k, I = cfg->moe_intermediate, Tm = cfg->max_tokens;
  const int64_t Tpad = (Tm + 127) / 128 * 128;
  const int64_t rows = Tpad + (Tm * k + E * 127 + 127) / 128 * 128;
  const int64_t xs_stride = (H / 128 + 3) / 4 * 4, hs_stride = (I / 128 + 3) / 4 * 4;
  plan->staging_slots = n_stage;
  plan->experts_per_launch = epl;
  const int64_t En = cfg->expert_end == 0 ? E : cfg->expert_end - cfg->expert_begin;
  {  // the last group of a long call (>= 256 rows per expert) is launched in pieces of kTailExperts experts (prefill_impl)
    const int groups = (En + epl - 1) / epl, last = En - (groups - 1) * epl;
    const bool pieces = last > kTailExperts && static_cast<long long>(cfg->max_tokens) * cfg->top_k >= 256LL * cfg->n_experts;
    const int last_launches = pieces ? (last + kTailExperts - 1) / kTailExperts : 1;
    plan->launch_pairs_streamed = static_cast<int32_t>(groups - 1 + last_launches + (cfg->n_shared ? 1 : 0));
  }
  plan->workspace_rows = rows;
  plan->expert_slot_bytes = 3 * I * H;
  plan->routed_bytes_per_pass = En * 3 * I * H;
  plan->pool_bytes_streamed = (1 + n_stage) * 3 * I * H;
  plan->pool_bytes_resident = (1 + En) * 3 * I * H;
  plan->scale_bytes = (E + 1) * (2 * (I / 128) * (H / 128) + (H / 128) * (I / 128)) * 4;
  plan->workspace_bytes = rows * (H + xs_stride * 4 + I + hs_stride * 4 + H * 2 + xs_stride * 4 + 4) + Tm * (E * 4 + k * 12);
  plan->fp8_flops_per_token = 2 * 3 * I * H * (k + cfg->n_shared);
  plan->gemm_smem_bytes_gateup = slp::tc::Cfg<0, false>::kSmemBytes;
  plan->gemm_smem_bytes_down = slp::tc::Cfg<1, false>::kSmemBytes;
  return SLP_OK;
}

slp_status slp_moe_set_residency(slp_moe_layer* h, slp_residency r) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  if (r != SLP_STREAMED && r != SLP_RESIDENT) return fail(SLP_ERR_INVALID_ARG, "unknown residency %d", static_cast<int>(r));
  CU_TRY(cudaSetDevice(h->cfg.device));
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  CU_TRY(cudaDeviceSynchronize());
  if (h->dead) return fail(SLP_ERR_OOM, "handle lost its expert pool in an earlier failed residency switch; destroy it");
  auto upload_all = [&]() -> slp_status {
    h->stats = slp_moe_stats{};
    slp_status u = copy_experts(h, h->e0, h->e1, nullptr);
    if (u != SLP_OK) return u;
    CU_TRY(cudaStreamSynchronize(h->copy_stream));
    h->pool_needs_upload = false;
    return SLP_OK;
  };
  if (static_cast<int>(r) == h->residency) {
    if (r == SLP_RESIDENT && h->pool_needs_upload) return upload_all();
    return SLP_OK;
  }
  if (r == SLP_RESIDENT && h->layers.size() > 1)
    return fail(SLP_ERR_UNSUPPORTED_SHAPE, "resident mode needs a single-layer handle (this stack has %zu layers sharing one ring)", h->layers.size());
  select_layer(h, 0);
  if (r == SLP_RESIDENT) {
    st = alloc_pool(h, h->e1 - h->e0, h->e1 - h->e0);
    if (st != SLP_OK) return st;   // the handle is unchanged (still streamed) unless it reports itself dead
    st = upload_all();
    if (st != SLP_OK) return st;
  } else {
    const int En = h->e1 - h->e0;
    int n_stage = h->cfg.staging_slots == 0 ? En : std::min(h->cfg.staging_slots, En);
    int epl = h->cfg.experts_per_launch;
    if (epl == 0) epl = auto_epl(n_stage, En);
    st = alloc_pool(h, n_stage, epl);
    if (st != SLP_OK) {
      // still resident; if the pool had to be rebuilt on the way back its experts are uploaded again
      if (!h->dead && h->pool_needs_upload) upload_all();
      return st;
    }
  }
  h->residency = r;
  return SLP_OK;
}

slp_status slp_moe_prefill(slp_moe_layer* h, const void* hidden_bf16, int32_t T, void* out_bf16, void* cuda_stream) {
  return slp_moe_stack_prefill(h, 0, hidden_bf16, T, out_bf16, cuda_stream);
}

slp_status slp_moe_stack_prefetch(slp_moe_layer* h, int32_t layer) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  if (layer < 0 || layer >= static_cast<int>(h->layers.size())) return fail(SLP_ERR_INVALID_ARG, "layer %d outside 0..%zu", layer, h->layers.size() - 1);
  if (h->dead) return fail(SLP_ERR_OOM, "handle lost its expert pool in an earlier failed residency switch; destroy it");
  CU_TRY(cudaSetDevice(h->cfg.device));
  const slp_moe_stats keep = h->stats;   // a bare prefetch is not a call: it leaves the last call's statistics alone
  slp_status st = prefetch_layer(h, layer);
  h->stats = keep;
  return st;
}

slp_status slp_moe_stack_prefill(slp_moe_layer* h, int32_t layer, const void* hidden_bf16, int32_t T, void* out_bf16, void* cuda_stream) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  if (layer < 0 || layer >= static_cast<int>(h->layers.size())) return fail(SLP_ERR_INVALID_ARG, "layer %d outside 0..%zu", layer, h->layers.size() - 1);
  if (T < 0 || T > h->Tm) return fail(SLP_ERR_INVALID_ARG, "T = %d outside 0..max_tokens (%d)", T, h->Tm);
  if (T == 0) return SLP_OK;
  if (!hidden_bf16 || !out_bf16) return fail(SLP_ERR_INVALID_ARG, "NULL hidden/out");
  if (hidden_bf16 == out_bf16) return fail(SLP_ERR_INVALID_ARG, "out must not alias hidden");
  CU_TRY(cudaSetDevice(h->cfg.device));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (h->dead) return fail(SLP_ERR_OOM, "handle lost its expert pool in an earlier failed residency switch; destroy it");
  if (h->in_flight) {
    cudaError_t q = cudaEventQuery(h->ev_done);
    if (q == cudaSuccess) {
      h->in_flight = false;
      slp_status ke = check_kernel_error(h);  // the previous call finished: did one of its kernels hit the watchdog?
      if (ke != SLP_OK) return ke;
    } else if (q == cudaErrorNotReady) {
      if (s != h->last_stream) return fail(SLP_ERR_BUSY, "a call is still in flight on another stream");
    } else {
      return fail(SLP_ERR_CUDA, "cudaEventQuery failed: %s", cudaGetErrorString(q));
    }
  }
  if (h->e0 != 0 || h->e1 != h->E)
    return fail(SLP_ERR_INVALID_ARG, "this handle owns experts [%d, %d) of %d: use slp_moe_prefill_partial and reduce the partial sums", h->e0, h->e1, h->E);
  return prefill_impl(h, hidden_bf16, T, out_bf16, s, false, 0, -1, layer);
}

slp_status slp_moe_prefill_partial(slp_moe_layer* h, const void* hidden_bf16, int32_t T, float* partial_f32, int32_t sh_t0, int32_t sh_t1,
                                   void* cuda_stream) {
  return slp_moe_stack_prefill_partial(h, 0, hidden_bf16, T, partial_f32, sh_t0, sh_t1, cuda_stream);
}

slp_status slp_moe_stack_prefill_partial(slp_moe_layer* h, int32_t layer, const void* hidden_bf16, int32_t T, float* partial_f32,
                                         int32_t sh_t0, int32_t sh_t1, void* cuda_stream) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  if (layer < 0 || layer >= static_cast<int>(h->layers.size())) return fail(SLP_ERR_INVALID_ARG, "layer %d outside 0..%zu", layer, h->layers.size() - 1);
  if (T < 0 || T > h->Tm) return fail(SLP_ERR_INVALID_ARG, "T = %d outside 0..max_tokens (%d)", T, h->Tm);
  if (T == 0) return SLP_OK;
  if (!hidden_bf16 || !partial_f32) return fail(SLP_ERR_INVALID_ARG, "NULL hidden/partial");
  if (sh_t0 < 0 || sh_t1 < sh_t0 || sh_t1 > T) return fail(SLP_ERR_INVALID_ARG, "shared token range [%d, %d) outside 0..%d", sh_t0, sh_t1, T);
  CU_TRY(cudaSetDevice(h->cfg.device));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (h->dead) return fail(SLP_ERR_OOM, "handle lost its expert pool in an earlier failed residency switch; destroy it");
  if (h->in_flight) {
    cudaError_t q = cudaEventQuery(h->ev_done);
    if (q == cudaSuccess) {
      h->in_flight = false;
      slp_status ke = check_kernel_error(h);
      if (ke != SLP_OK) return ke;
    } else if (q == cudaErrorNotReady) {
      if (s != h->last_stream) return fail(SLP_ERR_BUSY, "a call is still in flight on another stream");
    } else {
      return fail(SLP_ERR_CUDA, "cudaEventQuery failed: %s", cudaGetErrorString(q));
    }
  }
  return prefill_impl(h, hidden_bf16, T, partial_f32, s, true, sh_t0, sh_t1, layer);
}

slp_status slp_moe_finalize_partial(int32_t device, const float* sum_f32, size_t n_elems, void* out_bf16, void* cuda_stream) {
  if (!sum_f32 || !out_bf16) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  if (n_elems % 4) return fail(SLP_ERR_INVALID_ARG, "n_elems must be a multiple of 4");
  if (n_elems == 0) return SLP_OK;
  CU_TRY(cudaSetDevice(device));
  const size_t n4 = n_elems / 4;
  const int blocks = static_cast<int>(std::min<size_t>((n4 + 255) / 256, 148 * 16));
  slp::partial_to_bf16_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(sum_f32, static_cast<__nv_bfloat16*>(out_bf16), n4);
  CU_TRY(cudaGetLastError());
  return SLP_OK;
}

slp_status slp_moe_prefill_host(slp_moe_layer* h, const void* hidden_host, int32_t T, void* out_host) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  if (T < 0 || T > h->Tm) return fail(SLP_ERR_INVALID_ARG, "T = %d outside 0..max_tokens (%d)", T, h->Tm);
  if (T == 0) return SLP_OK;
  if (!hidden_host || !out_host) return fail(SLP_ERR_INVALID_ARG, "NULL hidden/out");
  if (h->e0 != 0 || h->e1 != h->E) return fail(SLP_ERR_INVALID_ARG, "expert-sharded handle: use slp_moe_prefill_partial");
  CU_TRY(cudaSetDevice(h->cfg.device));
  if (h->dead) return fail(SLP_ERR_OOM, "handle lost its expert pool in an earlier failed residency switch; destroy it");
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  const size_t bytes = static_cast<size_t>(h->Tm) * h->H * 2;
  if (!h->d_e2e_in) {
    CU_TRY(cudaMalloc(&h->d_e2e_in, bytes));
    CU_TRY(cudaMalloc(&h->d_e2e_out, bytes));
  }
  const size_t n = static_cast<size_t>(T) * h->H * 2;
  CU_TRY(cudaMemcpyAsync(h->d_e2e_in, hidden_host, n, cudaMemcpyHostToDevice, h->own_stream));
  st = prefill_impl(h, h->d_e2e_in, T, h->d_e2e_out, h->own_stream);
  if (st != SLP_OK) return st;
  CU_TRY(cudaMemcpyAsync(out_host, h->d_e2e_out, n, cudaMemcpyDeviceToHost, h->own_stream));
  CU_TRY(cudaStreamSynchronize(h->own_stream));
  h->in_flight = false;
  return check_kernel_error(h);
}

slp_status slp_moe_layer_destroy(slp_moe_layer* h) {
  if (!h) return SLP_OK;
  cudaSetDevice(h->cfg.device);
  cudaDeviceSynchronize();
  const slp_status guard_status = check_guards(h);  // reported by destroy too (triage "guards")
  free_pool(h);
  if (h->cur_layer >= 0 && h->cur_layer < static_cast<int>(h->layers.size())) stash_layer(h, h->cur_layer);
  for (LayerW& w : h->layers) {
    void* lp[] = {w.d_router_hl, w.d_router_w, w.d_bias, w.d_gate_s, w.d_up_s, w.d_down_s, w.d_shpool};
    for (void* p : lp)
      if (p) cudaFree(p);
  }
  void* ptrs[] = {h->d_logits, h->d_w, h->d_xs, h->d_hs, h->d_idx,
                  h->d_counts, h->d_chunk, h->d_row_start, h->d_tile_start, h->d_tile_expert, h->d_pair_start, h->d_pair_expert, h->d_tile_info, h->d_pos, h->d_row_token, h->d_xq,
                  h->d_hq, h->d_y, h->d_ys, h->d_err, h->d_clk, h->d_sched, h->d_e2e_in, h->d_e2e_out};
  for (void* p : ptrs) ws_free(h, p);
  if (h->h_counts) cudaFreeHost(h->h_counts);
  if (h->h_err) cudaFreeHost(h->h_err);
  for (void* p : h->registered) unregister_host_range(p);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  if (h->ev_done) cudaEventDestroy(h->ev_done);
  for (auto e : h->ev_t)
    if (e) cudaEventDestroy(e);
  if (h->ev_copy0) cudaEventDestroy(h->ev_copy0);
  if (h->ev_copy1) cudaEventDestroy(h->ev_copy1);
  for (auto e : h->ev_k)
    if (e) cudaEventDestroy(e);
  for (auto e : h->ev_tail)
    if (e) cudaEventDestroy(e);
  cudaGetLastError();
  delete h;
  return guard_status;
}

slp_status slp_moe_debug_routing(slp_moe_layer* h, int32_t* idx, float* w, int32_t* counts) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  CU_TRY(cudaSetDevice(h->cfg.device));
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  const size_t n = static_cast<size_t>(h->last_T) * h->k;
  if (idx) CU_TRY(cudaMemcpy(idx, h->d_idx, n * sizeof(int32_t), cudaMemcpyDeviceToHost));
  if (w) CU_TRY(cudaMemcpy(w, h->d_w, n * sizeof(float), cudaMemcpyDeviceToHost));
  if (counts) CU_TRY(cudaMemcpy(counts, h->d_counts, h->E * sizeof(int32_t), cudaMemcpyDeviceToHost));
  return check_kernel_error(h);
}

slp_status slp_moe_debug_quant_hidden(slp_moe_layer* h, uint8_t* xq, float* xs) {
  if (!h) return fail(SLP_ERR_INVALID_ARG, "NULL handle");
  CU_TRY(cudaSetDevice(h->cfg.device));
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  const int T = h->last_T;
  if (xq) CU_TRY(cudaMemcpy(xq, h->d_xq, static_cast<size_t>(T) * h->H, cudaMemcpyDeviceToHost));
  if (xs)
    CU_TRY(cudaMemcpy2D(xs, h->kbH * sizeof(float), h->d_xs, h->xs_stride * sizeof(float), h->kbH * sizeof(float), T, cudaMemcpyDeviceToHost));
  return check_kernel_error(h);
}

namespace {
// device address and size (for the last call) of a debug buffer
slp_status locate_buffer(slp_moe_layer* h, int32_t which, const void** src, size_t* size) {
  int32_t rs[1] = {0};  // row_start[E+1] = rows in use
  CU_TRY(cudaMemcpy(rs, h->d_row_start + h->E + 1, sizeof(int32_t), cudaMemcpyDeviceToHost));
  const size_t rows = static_cast<size_t>(rs[0]), T = h->last_T;
  switch (which) {
    case SLP_BUF_COUNTS: *src = h->d_counts; *size = h->E * sizeof(int32_t); break;
    case SLP_BUF_ROW_START: *src = h->d_row_start; *size = (h->E + 1) * sizeof(int32_t); break;
    case SLP_BUF_POS: *src = h->d_pos; *size = T * h->k * sizeof(int32_t); break;
    case SLP_BUF_ROW_TOKEN: *src = h->d_row_token; *size = rows * sizeof(int32_t); break;
    case SLP_BUF_HQ: *src = h->d_hq; *size = rows * h->I; break;
    case SLP_BUF_HS: *src = h->d_hs; *size = rows * h->hs_stride * sizeof(float); break;
    case SLP_BUF_Y: *src = h->d_y; *size = rows * h->H * sizeof(uint16_t); break;
    case SLP_BUF_LOGITS: *src = h->d_logits; *size = T * h->E * sizeof(float); break;
    case SLP_BUF_YS: *src = h->d_ys; *size = rows * h->ys_stride * sizeof(float); break;
    default: return fail(SLP_ERR_INVALID_ARG, "unknown buffer id %d", which);
  }
  return SLP_OK;
}
}  // namespace

slp_status slp_moe_debug_buffer(slp_moe_layer* h, int32_t which, void* dst, size_t bytes, size_t* written) {
  if (!h || !dst) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  CU_TRY(cudaSetDevice(h->cfg.device));
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  const void* src = nullptr;
  size_t size = 0;
  st = locate_buffer(h, which, &src, &size);
  if (st != SLP_OK) return st;
  const size_t n = std::min(size, bytes);
  if (n) CU_TRY(cudaMemcpy(dst, src, n, cudaMemcpyDeviceToHost));
  if (written) *written = size;
  return check_kernel_error(h);
}

slp_status slp_moe_debug_buffer_range(slp_moe_layer* h, int32_t which, size_t offset, size_t bytes, void* dst) {
  if (!h || !dst) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  CU_TRY(cudaSetDevice(h->cfg.device));
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  const void* src = nullptr;
  size_t size = 0;
  st = locate_buffer(h, which, &src, &size);
  if (st != SLP_OK) return st;
  if (offset > size || bytes > size - offset) return fail(SLP_ERR_INVALID_ARG, "range [%zu, +%zu) leaves the buffer of %zu bytes", offset, bytes, size);
  if (bytes) CU_TRY(cudaMemcpy(dst, static_cast<const char*>(src) + offset, bytes, cudaMemcpyDeviceToHost));
  return check_kernel_error(h);
}

slp_status slp_moe_get_stats(slp_moe_layer* h, slp_moe_stats* stats) {
  if (!h || !stats) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  if (stats->struct_size != sizeof(slp_moe_stats)) return fail(SLP_ERR_INVALID_ARG, "stats.struct_size mismatch");
  CU_TRY(cudaSetDevice(h->cfg.device));
  slp_status st = wait_idle(h);
  if (st != SLP_OK) return st;
  if (h->last_T > 0) {
    CU_TRY(cudaEventSynchronize(h->ev_t[4]));
    CU_TRY(cudaEventElapsedTime(&h->stats.ms_total, h->ev_t[0], h->ev_t[4]));
    CU_TRY(cudaEventElapsedTime(&h->stats.ms_route, h->ev_t[0], h->ev_t[1]));
    CU_TRY(cudaEventElapsedTime(&h->stats.ms_experts, h->ev_t[2], h->ev_t[3]));
    CU_TRY(cudaEventElapsedTime(&h->stats.ms_combine, h->ev_t[3], h->ev_t[4]));
    if (h->stats_copy_valid) {
      CU_TRY(cudaEventSynchronize(h->ev_copy1));
      CU_TRY(cudaEventElapsedTime(&h->stats.ms_copy_span, h->ev_copy0, h->ev_copy1));
    }
    h->stats.ms_gateup_sum = h->stats.ms_down_sum = h->stats.ms_gateup_shared = h->stats.ms_down_shared = 0.f;
    h->stats.timed_gemm_pairs = h->ev_k_used / 3;
    for (int i = 0; i + 3 <= h->ev_k_used; i += 3) {
      float a = 0.f, b = 0.f;
      CU_TRY(cudaEventElapsedTime(&a, h->ev_k[i], h->ev_k[i + 1]));
      CU_TRY(cudaEventElapsedTime(&b, h->ev_k[i + 1], h->ev_k[i + 2]));
      h->stats.ms_gateup_sum += a;
      h->stats.ms_down_sum += b;
      if (i == h->ev_k_shared) {
        h->stats.ms_gateup_shared = a;
        h->stats.ms_down_shared = b;
      }
    }
    unsigned long long clk[16] = {};
    CU_TRY(cudaMemcpy(clk, h->d_clk, sizeof clk, cudaMemcpyDeviceToHost));
#ifdef SLP_PROF
    for (int m = 0; m < 2; ++m)
      if (clk[7 + 4 * m])
        fprintf(stderr, "[slp prof] mode %d: tiles/CTA-warp0 %llu, per tile: next tile + scale prefetch %.0f, first-wait %.0f, K loop %.0f, epilogue %.0f cycles\n", m,
                clk[7 + 4 * m], double(clk[12 + m]) / clk[7 + 4 * m], double(clk[4 + 4 * m]) / clk[7 + 4 * m], double(clk[5 + 4 * m]) / clk[7 + 4 * m], double(clk[6 + 4 * m]) / clk[7 + 4 * m]);
#endif
    h->stats.sm_mhz_gateup = clk[1] ? static_cast<float>(1e3 * static_cast<double>(clk[0]) / static_cast<double>(clk[1])) : 0.f;
    h->stats.sm_mhz_down = clk[3] ? static_cast<float>(1e3 * static_cast<double>(clk[2]) / static_cast<double>(clk[3])) : 0.f;
    int32_t ts[1] = {0};
    CU_TRY(cudaMemcpy(ts, h->d_tile_start + h->E + 1, sizeof(int32_t), cudaMemcpyDeviceToHost));
    h->stats.m_tiles = ts[0];
  }
  *stats = h->stats;
  stats->struct_size = sizeof(slp_moe_stats);
  slp_status gst = check_guards(h);
  if (gst != SLP_OK) return gst;
  return check_kernel_error(h);
}

slp_status slp_measure_h2d(int32_t device, size_t chunk_bytes, size_t total_bytes, int32_t repeats, double* gbs) {
  if (!gbs || chunk_bytes == 0 || total_bytes < chunk_bytes || repeats <= 0) return fail(SLP_ERR_INVALID_ARG, "bad arguments");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
    cudaGetLastError();
    return fail(SLP_ERR_CUDA, "no such CUDA device %d", device);
  }
  CU_TRY(cudaSetDevice(device));
  const size_t n_chunks = total_bytes / chunk_bytes;
  void *hbuf = nullptr, *dbuf = nullptr;
  cudaStream_t s = nullptr;
  cudaEvent_t a = nullptr, b = nullptr;
  CU_TRY(cudaMallocHost(&hbuf, n_chunks * chunk_bytes));
  memset(hbuf, 1, n_chunks * chunk_bytes);
  slp_status st = SLP_OK;
  double best = 0;
  if (cudaMalloc(&dbuf, n_chunks * chunk_bytes) != cudaSuccess || cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
    st = fail(SLP_ERR_CUDA, "setup failed: %s", cudaGetErrorString(cudaGetLastError()));
  } else {
    for (int r = 0; r < repeats + 1 && st == SLP_OK; ++r) {
      cudaEventRecord(a, s);
      for (size_t c = 0; c < n_chunks; ++c)
        cudaMemcpyAsync(static_cast<char*>(dbuf) + c * chunk_bytes, static_cast<char*>(hbuf) + c * chunk_bytes, chunk_bytes,
                        cudaMemcpyHostToDevice, s);
      cudaEventRecord(b, s);
      if (cudaEventSynchronize(b) != cudaSuccess) {
        st = fail(SLP_ERR_CUDA, "copy failed: %s", cudaGetErrorString(cudaGetLastError()));
        break;
      }
      float ms = 0;
      cudaEventElapsedTime(&ms, a, b);
      if (r > 0) best = std::max(best, static_cast<double>(n_chunks * chunk_bytes) / (ms * 1e-3) / 1e9);
    }
  }
  if (a) cudaEventDestroy(a);
  if (b) cudaEventDestroy(b);
  if (s) cudaStreamDestroy(s);
  if (dbuf) cudaFree(dbuf);
  cudaFreeHost(hbuf);
  *gbs = best;
  return st;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// slp_moe_permute_static (include/slp_moe.h): the histogram / scan / permute step (a2) for callers
// that are not allowed to allocate device memory.
//
// Who that is: code that runs inside somebody else's memory budget.  An inference server that
// hands the whole HBM to its own pool allocator at start-up, a plugin called from inside a region
// the host framework has frozen (a stream capture, a real-time loop with a no-driver-allocation
// rule), or a process started with the device already full: for all of them cudaMalloc either
// fails, stalls the device behind an implicit synchronisation, or is forbidden outright.  The
// handle-based calls above allocate at create; this one needs no handle and allocates nothing,
// ever: the only memory it uses beyond the caller's inputs and outputs is the array below, which
// is part of the library image and is placed in device memory by the CUDA runtime when the
// library is loaded on a GPU.  The price is that every GPU the process touches through this
// library holds kStaticScratchBytes until the process exits, and that the sizes are capped.
//
// g_static_scratch is a DEVICE variable.  On the host its name is only a handle for the runtime
// (it has a host-side shadow address that no GPU can use), so host code must never pass it to a
// kernel directly.  The device address is asked for once per device, with that device current,
// through cudaGetSymbolAddress, and it is that pointer the kernels receive.
// ---------------------------------------------------------------------------------------------
namespace slp_static {
constexpr int kMaxTokens = 32768;         // T
constexpr int kMaxAssignments = 262144;   // T * top_k (32768 tokens x top-8)
constexpr int kMaxTiles = 4096;           // >= Tpad/128 + T*k/128 + E + 2 at the limits above (256 + 2048 + 511 + 2)
constexpr int kMaxDevices = 64;
// byte offsets of the pieces inside the array (all multiples of 256)
constexpr size_t kOffChunk = 0;                                                                    // int32 [256 chunks][E]
constexpr size_t kOffTileInfo = kOffChunk + (kMaxTokens / slp::kChunkTokens) * slp::kMaxExperts * sizeof(int32_t);
constexpr size_t kOffTileExpert = kOffTileInfo + kMaxTiles * sizeof(int4);
constexpr size_t kOffPairExpert = kOffTileExpert + kMaxTiles * sizeof(int32_t);
constexpr size_t kOffTileStart = kOffPairExpert + kMaxTiles * sizeof(int32_t);
constexpr size_t kOffPairStart = kOffTileStart + 4096;
constexpr size_t kStaticScratchBytes = kOffPairStart + 4096;                                       // 630 784 B = 616 KiB
static_assert(kOffTileInfo % 256 == 0 && kOffTileExpert % 256 == 0 && kOffPairExpert % 256 == 0 && kOffTileStart % 256 == 0 &&
              kOffPairStart % 256 == 0, "pieces of the static scratch must stay 256-byte aligned");
static_assert((slp::kMaxExperts + 2) * sizeof(int32_t) <= 4096, "tile_start / pair_start piece too small");
}  // namespace slp_static

static __device__ __align__(256) unsigned char g_static_scratch[slp_static::kStaticScratchBytes];

namespace slp_static {
std::mutex g_mutex;
unsigned char* g_dev_ptr[kMaxDevices] = {};  // device address of g_static_scratch on each device, once looked up

// First use on `device` (which must be current): ask the runtime where this device's copy of the array lives.
slp_status scratch_for_device(int device, unsigned char** out) {
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_dev_ptr[device]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return fail(SLP_ERR_CUDA, "cudaGetSymbolAddress(g_static_scratch) on device %d failed: %s", device, cudaGetErrorString(e));
    }
    g_dev_ptr[device] = static_cast<unsigned char*>(p);
  }
  *out = g_dev_ptr[device];
  return SLP_OK;
}
}  // namespace slp_static

extern "C" int64_t slp_moe_permute_static_rows(int32_t T, int32_t top_k, int32_t n_experts) {
  if (T < 0 || top_k < 0 || n_experts < 0) return -1;
  const int64_t Tpad = (static_cast<int64_t>(T) + 127) / 128 * 128;
  return Tpad + (static_cast<int64_t>(T) * top_k + static_cast<int64_t>(n_experts) * 127 + 127) / 128 * 128;
}

extern "C" slp_status slp_moe_permute_static(int32_t device, const int32_t* idx_dev, int32_t T, int32_t top_k, int32_t n_experts,
                                             int32_t* counts_dev, int32_t* row_start_dev, int32_t* pos_dev, int32_t* row_token_dev,
                                             int64_t row_capacity, void* cuda_stream) {
  namespace st = slp_static;
  const int E = n_experts, k = top_k;
  if (E <= 0 || E > slp::kMaxExperts - 1) return fail(SLP_ERR_UNSUPPORTED_SHAPE, "n_experts %d outside 1..%d", E, slp::kMaxExperts - 1);
  if (k <= 0 || k > 32 || k > E) return fail(SLP_ERR_UNSUPPORTED_SHAPE, "top_k %d outside 1..min(32, n_experts)", k);
  if (T < 0 || T > st::kMaxTokens)
    return fail(SLP_ERR_UNSUPPORTED_SHAPE, "T = %d exceeds the static scratch of slp_moe_permute_static (at most %d tokens per call)", T, st::kMaxTokens);
  if (static_cast<int64_t>(T) * k > st::kMaxAssignments)
    return fail(SLP_ERR_UNSUPPORTED_SHAPE, "T * top_k = %lld exceeds the static scratch of slp_moe_permute_static (at most %d routed assignments per call)",
                static_cast<long long>(T) * k, st::kMaxAssignments);
  if (T == 0) return SLP_OK;
  if (!idx_dev || !counts_dev || !row_start_dev || !pos_dev || !row_token_dev) return fail(SLP_ERR_INVALID_ARG, "NULL argument");
  const int64_t rows_bound = slp_moe_permute_static_rows(T, k, E);
  if (row_capacity < rows_bound)
    return fail(SLP_ERR_INVALID_ARG, "row_capacity %lld below slp_moe_permute_static_rows(T, top_k, n_experts) = %lld",
                static_cast<long long>(row_capacity), static_cast<long long>(rows_bound));
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev || device >= st::kMaxDevices) {
    cudaGetLastError();
    return fail(SLP_ERR_CUDA, "no such CUDA device %d", device);
  }
  CU_TRY(cudaSetDevice(device));
  unsigned char* base = nullptr;
  slp_status rc = st::scratch_for_device(device, &base);
  if (rc != SLP_OK) return rc;
  int32_t* chunk = reinterpret_cast<int32_t*>(base + st::kOffChunk);
  int4* tile_info = reinterpret_cast<int4*>(base + st::kOffTileInfo);
  int32_t* tile_expert = reinterpret_cast<int32_t*>(base + st::kOffTileExpert);
  int32_t* pair_expert = reinterpret_cast<int32_t*>(base + st::kOffPairExpert);
  int32_t* tile_start = reinterpret_cast<int32_t*>(base + st::kOffTileStart);
  int32_t* pair_start = reinterpret_cast<int32_t*>(base + st::kOffPairStart);

  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int n_chunks = (T + slp::kChunkTokens - 1) / slp::kChunkTokens;
  const int wpb = 4;
  const int blocks = (n_chunks + wpb - 1) / wpb;
  const size_t sm = static_cast<size_t>(wpb) * E * sizeof(int32_t);
  // The array still holds whatever the previous call left there.  Nothing in it has to start at zero: the histogram pass
  // stores (not adds) all E counters of each of this call's n_chunks chunks before the scan reads them, and the scan
  // writes every table entry the place pass reads.  What does need a known start value is the caller's row_token (-1 in
  // the padding rows of every expert range), so that is filled here.
  CU_TRY(cudaMemsetAsync(row_token_dev, 0xFF, static_cast<size_t>(rows_bound) * sizeof(int32_t), s));
  slp::permute_hist_kernel<<<blocks, wpb * 32, sm, s>>>(idx_dev, chunk, T, k, E);
  slp::permute_scan_kernel<<<1, 512, 0, s>>>(chunk, counts_dev, row_start_dev, tile_start, tile_expert, pair_start, pair_expert, tile_info,
                                             n_chunks, T, E, 0, E, 0, T);
  slp::permute_place_kernel<<<blocks, wpb * 32, sm, s>>>(idx_dev, chunk, row_start_dev, pos_dev, row_token_dev, T, k, E, 0, E);
  CU_TRY(cudaGetLastError());
  return SLP_OK;
}
