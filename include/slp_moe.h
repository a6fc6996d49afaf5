/* slp_moe.h — C ABI of libslpmoe: one routed-MoE layer of stream-loading prefill (SLP) on one B200.
 *
 * The problem, as the paper states it: a layer's FP8 expert weights live in pinned host DRAM (the
 * authoritative copy never leaves the host, §3.1 "the authoritative copy always
 * remains in host memory"); a prompt chunk's hidden states are on the GPU; the module is executed
 * on a stream in order with other modules while a loader stages its weights into GPU memory and
 * signals readiness with events (§3.1, Fig. 5).  The module itself is
 * gate -> sort -> expert FFNs -> weighted sum (Fig. 2 steps 3-5; PAPER.md:48 shared
 * experts; Fig. 11 gate/up/down), on FP8 weights with block scales, activations
 * quantised to FP8, FP32 accumulation (§2.2.5, PAPER.md:235,255 128-wide K blocks).
 *
 * Every step runs in hand-written CUDA kernels for sm_100a.  There is no CPU path: every entry
 * point that needs the GPU returns SLP_ERR_CUDA when none is usable.
 *
 * Conventions
 *  - All functions return slp_status (0 = ok, negative = error); slp_last_error() returns a
 *    thread-local, NUL-terminated description of the last error on the calling thread.
 *    No C++ exception crosses this boundary.
 *  - "host" pointers are CPU addresses, "dev" pointers are CUDA device addresses on cfg.device.
 *  - Tensors are dense row-major.  bf16 = 16-bit brain float bit patterns.  e4m3 = OCP FP8 E4M3
 *    (bias 7, max 448, 0x7F/0xFF = NaN, no infinities).
 *  - Shapes: hidden H and moe_intermediate I are multiples of 128; n_experts E divisible by
 *    n_group; 1 <= top_k <= 32, top_k <= topk_group * E / n_group; E <= 512; n_shared in {0, 1}
 *    with shared_intermediate == moe_intermediate.  Anything else: SLP_ERR_UNSUPPORTED_SHAPE at
 *    create (never a silent fallback).
 */
#ifndef SLP_MOE_H
#define SLP_MOE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SLP_MOE_ABI_VERSION 3u /* layout and meaning of the structs below; checked by create and query_plan */

typedef struct slp_moe_layer slp_moe_layer; /* opaque handle */

typedef enum {
  SLP_OK = 0,
  SLP_ERR_INVALID_ARG = -1,
  SLP_ERR_UNSUPPORTED_SHAPE = -2,
  SLP_ERR_CUDA = -3,
  SLP_ERR_OOM = -4,
  SLP_ERR_NOT_PINNED = -5,
  SLP_ERR_BUSY = -6,
  SLP_ERR_KERNEL_TIMEOUT = -7 /* an in-kernel pipeline wait exceeded its watchdog bound */
} slp_status;

typedef enum { SLP_STREAMED = 0, SLP_RESIDENT = 1 } slp_residency;
typedef enum { SLP_SCORE_SIGMOID_BIAS = 0, SLP_SCORE_SOFTMAX = 1 } slp_scoring;

/* Layer configuration (PAPER.md:48 gate; BASELINE.json configs for the constants). */
typedef struct {
  uint32_t struct_size;       /* = sizeof(slp_moe_cfg); ABI versioning */
  int32_t device;             /* CUDA ordinal */
  int32_t hidden;             /* H */
  int32_t n_experts;          /* E routed experts */
  int32_t top_k;              /* k */
  int32_t n_group;            /* G contiguous expert groups (1 = no grouping) */
  int32_t topk_group;         /* groups kept per token */
  int32_t moe_intermediate;   /* I */
  int32_t n_shared;           /* 0 or 1 shared expert, always active, weight 1 */
  int32_t shared_intermediate;/* must equal moe_intermediate when n_shared == 1 */
  int32_t scoring;            /* slp_scoring */
  int32_t norm_topk;          /* 1: w_j = s_j / sum_j s_j * routed_scale; 0: w_j = s_j * routed_scale */
  float routed_scale;
  int32_t max_tokens;         /* workspace is sized for this T */
  int32_t staging_slots;      /* streamed mode: expert slots in HBM, the paper's ring length
                                 ("the number of experts of a layer" for short
                                 prompts, 2 = ping-pong for very long ones).  0 = auto (= E).
                                 Valid: 2..E. */
  int32_t experts_per_launch; /* streamed mode: experts whose tiles one GEMM launch covers once
                                 their copies have landed.  0 = auto.  Valid: 1..staging_slots/2
                                 (or staging_slots when staging_slots == E). */
  int32_t skip_empty_experts; /* 1: experts that received no token are neither copied nor run
                                 (needs the counts on the host: one small D2H + sync inside
                                 prefill).  0: paper-faithful fixed order, every expert copied. */
  int32_t require_pinned;     /* 1: create fails with SLP_ERR_NOT_PINNED if a weight buffer is
                                 pageable.  0: create pins it with cudaHostRegister. */
  int32_t expert_begin;       /* Expert sharding (the paper's SmallEP): this handle owns the routed */
  int32_t expert_end;         /* experts [expert_begin, expert_end).  0, 0 = all E.  A sharded handle still routes every
                                 token over all E experts, but copies, stores and runs only its own experts; the host
                                 pointers of the other experts may be NULL.  It is driven through
                                 slp_moe_prefill_partial; staging_slots counts this handle's experts. */
  uint32_t abi_version;       /* = SLP_MOE_ABI_VERSION of the header the caller was built with.  Fields of this struct
                                 have changed meaning in place before (gemm_impl / router_impl became expert_begin /
                                 expert_end at the same size); from ABI 3 on any such change bumps this number, and a
                                 caller built against an older header is refused (by struct_size: the field is new). */
} slp_moe_cfg;

/* Host weight pointers.  Borrowed for the lifetime of the handle; the host copy stays
 * authoritative.  Routed expert weights stay on the host in streamed mode and are
 * copied per call; router weights, bias, all fp32 block scales and the shared expert are uploaded
 * once by create and stay resident (BASELINE.json config 1: shared expert "kept resident"). */
typedef struct {
  const float* router_w;            /* [E, H] fp32 */
  const float* router_bias;         /* [E] fp32, or NULL (softmax scoring ignores it) */
  const uint8_t* const* gate_q;     /* E pointers, each [I, H] e4m3 (K = H contiguous) */
  const float* const* gate_s;       /* E pointers, each [I/128, H/128] fp32; w = decode(q) * s */
  const uint8_t* const* up_q;       /* as gate */
  const float* const* up_s;
  const uint8_t* const* down_q;     /* E pointers, each [H, I] e4m3 (K = I contiguous) */
  const float* const* down_s;       /* E pointers, each [H/128, I/128] fp32 */
  const uint8_t* shared_gate_q;     /* [I, H] or NULL when n_shared == 0 */
  const float* shared_gate_s;
  const uint8_t* shared_up_q;
  const float* shared_up_s;
  const uint8_t* shared_down_q;     /* [H, I] */
  const float* shared_down_s;
} slp_moe_host_weights;

/* Per-call statistics of the most recent completed slp_moe_prefill (CUDA-event times, ms). */
typedef struct {
  uint32_t struct_size;
  int32_t tokens;
  int32_t residency;
  int32_t experts_copied;
  int32_t experts_skipped;
  int64_t bytes_copied;       /* host -> HBM bytes moved by the streaming engine */
  float ms_total;             /* entry to exit on the caller's stream */
  float ms_copy_span;         /* first H2D start to last H2D end on the copy stream (0 if resident) */
  float ms_route;             /* router + histogram/scan/permute + hidden quantisation */
  float ms_experts;           /* first expert GEMM launch to last (includes waits on copies) */
  float ms_combine;
  int32_t gemm_launches;      /* grouped-GEMM kernel launches in the call */
  int32_t kernel_launches;    /* all kernel launches in the call */
  int32_t m_tiles;            /* 128-row tiles over all experts incl. shared */
  int32_t timed_gemm_pairs;   /* gate/up + down launch pairs bracketed by CUDA events on the caller's stream */
  float ms_gateup_sum;        /* sum over those launches of the gate/up (+SwiGLU+requant) kernel time */
  float ms_down_sum;          /* same for the down kernel */
  float sm_mhz_gateup;        /* average SM clock during the gate/up launches (clock64 / globaltimer of CTA 0) */
  float sm_mhz_down;          /* same for the down launches */
  int32_t h2d_copies;         /* cudaMemcpyAsync calls the streaming engine issued (consecutive experts merge) */
  int32_t experts_from_prefetch; /* experts of this call whose weights an earlier call had already prefetched (stacks) */
  int32_t experts_prefetched; /* experts of the NEXT layer whose copies this call enqueued ahead (stacks) */
  int32_t layer;              /* layer of the stack the call ran */
  int64_t bytes_prefetched;   /* host -> HBM bytes of those prefetch copies (not part of bytes_copied) */
  float ms_gateup_shared;     /* part of ms_gateup_sum spent in the shared expert's OWN launch (streamed mode launches it apart
                                 from the routed groups; 0 when it shares a launch with routed experts) */
  float ms_down_shared;       /* same for the down kernel */
} slp_moe_stats;

/* What create would allocate and how prefill would launch for a configuration (host arithmetic only). */
typedef struct {
  uint32_t struct_size;            /* = sizeof(slp_moe_plan) */
  int32_t staging_slots;           /* expert slots of the streamed ring after defaults (0 -> n_experts) */
  int32_t experts_per_launch;      /* experts per grouped-GEMM launch pair after defaults */
  int32_t launch_pairs_streamed;   /* gate/up + down launch pairs of a streamed call of max_tokens tokens (incl. the shared
                                      expert; with >= 256 rows per expert the last group of a call is launched in pieces
                                      of 8 experts to shorten the call's tail) */
  int64_t workspace_rows;          /* rows of xq / hq / Y: padded tokens + 128-aligned expert ranges */
  int64_t expert_slot_bytes;       /* 3 * I * H: gate | up | down of one expert ("3 FP8 linears") */
  int64_t routed_bytes_per_pass;   /* E * 3 * I * H: what one streamed call moves over the host link */
  int64_t pool_bytes_streamed;     /* (1 + staging_slots) slots */
  int64_t pool_bytes_resident;     /* (1 + E) slots */
  int64_t scale_bytes;             /* resident fp32 block scales of all experts */
  int64_t workspace_bytes;         /* activations and routing tables for max_tokens (approximate total) */
  int64_t fp8_flops_per_token;     /* 2 * 3 * I * H * (top_k + n_shared) */
  int32_t gemm_smem_bytes_gateup;  /* dynamic shared memory of the grouped-GEMM kernels */
  int32_t gemm_smem_bytes_down;
} slp_moe_plan;

/* Buffers readable through slp_moe_debug_buffer (parity / evidence; layouts in DESIGN.md §5). */
typedef enum {
  SLP_BUF_COUNTS = 0,      /* int32 [E] tokens per routed expert */
  SLP_BUF_ROW_START = 1,   /* int32 [E+1] first workspace row of each expert (entry E = shared) */
  SLP_BUF_POS = 2,         /* int32 [T, k] workspace row of (t, j) */
  SLP_BUF_ROW_TOKEN = 3,   /* int32 [rows] token id of each workspace row (-1 = padding) */
  SLP_BUF_HQ = 4,          /* uint8 [rows, I] requantised SwiGLU output */
  SLP_BUF_HS = 5,          /* float [rows, ceil4(I/128)] its scales */
  SLP_BUF_Y = 6,           /* fp16 [rows, H] per-row expert outputs (before the routing weights), block-scaled:
                              value = y16 * ys[row, column / 128] */
  SLP_BUF_LOGITS = 7,      /* float [T, E] router logits */
  SLP_BUF_YS = 8           /* float [rows, ceil4(H/128)] power-of-two scales of SLP_BUF_Y */
} slp_debug_buffer_id;

/* Create a layer.  Validates shapes, pins (or checks) the host weights, uploads the resident
 * tensors, allocates workspace for cfg->max_tokens and the expert slots.  Starts in SLP_STREAMED.
 * Errors: INVALID_ARG (NULL / bad struct_size), UNSUPPORTED_SHAPE, NOT_PINNED, OOM, CUDA. */
slp_status slp_moe_layer_create(const slp_moe_cfg* cfg, const slp_moe_host_weights* w, slp_moe_layer** out);

/* Multi-layer handle (Fig. 5: the loader walks the modules of successive layers while the model
 * thread executes them; "the experts ring buffer is shared across layers").  n_layers weight sets of the same shape
 * share ONE ring of expert slots, one workspace and one copy stream: the HBM cost of the streamed experts is
 * staging_slots slots however many layers there are, and no cudaMalloc / cudaFree happens after create.
 * `w` points to n_layers slp_moe_host_weights.  Router weights, biases, block scales and shared experts of all layers
 * are uploaded at create and stay resident.  slp_moe_layer_create is the n_layers == 1 case; every call that takes
 * a handle works on a stack (the single-layer calls address layer 0).  Resident mode needs n_layers == 1. */
slp_status slp_moe_stack_create(const slp_moe_cfg* cfg, int32_t n_layers, const slp_moe_host_weights* w, slp_moe_layer** out);

/* slp_moe_prefill on layer `layer` of a stack.  After enqueueing the layer's own work the loader keeps going: the
 * copies of layer (layer + 1) % n_layers are enqueued on the copy stream, each waiting only for the OFF event of
 * the ring slot it overwrites, so the next layer's experts stream in while this layer still computes and the next
 * call finds them loaded (or loading) instead of starting its weight pass from scratch.  n_layers == 1: no
 * prefetch.  Prefetched groups are always copied whole (routing of the next layer is not known yet). */
slp_status slp_moe_stack_prefill(slp_moe_layer* h, int32_t layer, const void* hidden_bf16, int32_t T, void* out_bf16, void* cuda_stream);

/* Explicit loader run-ahead: enqueue the copies of `layer` now (as many launch groups as the ring has slots that
 * hold no unconsumed prefetch of that same layer; an unconsumed prefetch of another layer is overwritten).  Returns
 * immediately; a later slp_moe_stack_prefill(layer) consumes them. */
slp_status slp_moe_stack_prefetch(slp_moe_layer* h, int32_t layer);

/* Validates cfg exactly as create does and fills *plan; needs no GPU and allocates nothing.
 * Errors: INVALID_ARG, UNSUPPORTED_SHAPE (same messages as create). */
slp_status slp_moe_query_plan(const slp_moe_cfg* cfg, slp_moe_plan* plan);

/* Switch residency.  SLP_RESIDENT uploads all E experts into HBM once (blocking) and later calls
 * copy nothing; SLP_STREAMED frees that copy and returns to per-call streaming.  Blocks until the
 * handle is idle. */
slp_status slp_moe_set_residency(slp_moe_layer* h, slp_residency r);

/* out[t,:] = sum_j w[t,j] * FFN_{idx[t,j]}(hidden[t,:]) + FFN_shared(hidden[t,:]), bf16, no residual.
 *  hidden_bf16: dev [T, H] bf16, read only.  out_bf16: dev [T, H] bf16, fully overwritten; must
 *  not alias hidden.  T in 0..max_tokens (T == 0 returns SLP_OK and touches nothing).
 *  cuda_stream: a cudaStream_t (0 = legacy default stream).  Asynchronous: every kernel of the call is
 *  ordered after prior work on cuda_stream and `out` is valid for later work on it.
 *  Copy stream (streamed mode): the host -> HBM expert copies run on the library's own copy stream.  They
 *  wait only for the ring slot they overwrite to be free (the OFF event of the launch that last used it,
 *  PAPER.md:138), NOT for prior work on cuda_stream: the weights do not depend on anything the caller
 *  computes, so the first copies of a call start as soon as the call is enqueued, and across back-to-back
 *  calls on one stream the next call's copies overlap the current call's last GEMMs (cross-call prefetch,
 *  the single-layer form of the paper's "load the next module while this one executes").  The kernels that
 *  consume a slot wait for its ON event, and the call's last record on cuda_stream follows all of them, so
 *  `out` ordering is unaffected.  The host weight buffers must not change while a handle borrows them.
 *  Calls in flight: calls on ONE stream may be enqueued back to back without waiting (they serialise on the
 *  stream and share the workspace safely); slp_moe_get_stats then describes the most recent call.  A call
 *  on a DIFFERENT stream while the previous call has not finished on the device returns SLP_ERR_BUSY (the
 *  workspace is per handle).  If the previous call has finished and one of its kernels hit the in-kernel
 *  watchdog, this call returns SLP_ERR_KERNEL_TIMEOUT and enqueues nothing.
 *  With skip_empty_experts == 1 the call synchronises cuda_stream once internally. */
slp_status slp_moe_prefill(slp_moe_layer* h, const void* hidden_bf16, int32_t T, void* out_bf16, void* cuda_stream);

/* SmallEP step 2-4 on one rank ("every rank gates and sorts the full batch locally and keeps only
 * tokens for its local experts ... executes its local experts and produces a partial weighted sum of shape [N, D]").
 *  hidden_bf16: dev [T, H], the ALL-GATHERED hidden states of all ranks (same on every rank).
 *  partial_f32: dev [T, H] fp32, fully overwritten with  sum over this handle's experts of w[t,j] * FFN(hidden[t])
 *  for every token, plus FFN_shared(hidden[t]) for tokens t in [shared_token_begin, shared_token_end) only (the
 *  shared expert is token-sharded; an empty range leaves it out; the range may start and end at any token: internally
 *  the shared expert's GEMMs start at shared_token_begin rounded down to a multiple of 32, which is what
 *  SLP_BUF_ROW_START[E] then reports, and the extra rows are never added to anything).  No bf16 rounding: the ranks' partial sums are
 *  added first (reduce-scatter) and rounded once by slp_moe_finalize_partial.  Works on an unsharded handle too
 *  (then the partial sum is the whole layer in fp32).  Ordering, copy stream and error rules as slp_moe_prefill. */
slp_status slp_moe_prefill_partial(slp_moe_layer* h, const void* hidden_bf16, int32_t T, float* partial_f32,
                                   int32_t shared_token_begin, int32_t shared_token_end, void* cuda_stream);

/* slp_moe_prefill_partial on layer `layer` of a stack (slp_moe_prefill_partial itself addresses layer 0), with the same
 * run-ahead of layer (layer + 1) % n_layers as slp_moe_stack_prefill: SmallEP over a multi-layer, expert-sharded stack.
 * INVALID_ARG for a layer outside the stack. */
slp_status slp_moe_stack_prefill_partial(slp_moe_layer* h, int32_t layer, const void* hidden_bf16, int32_t T, float* partial_f32,
                                         int32_t shared_token_begin, int32_t shared_token_end, void* cuda_stream);

/* out_bf16[i] = bf16_rne(sum_f32[i]) for n_elems elements (multiple of 4) on `device`: the single output rounding
 * of the SmallEP path, applied to the reduce-scattered sum.  Asynchronous on cuda_stream. */
slp_status slp_moe_finalize_partial(int32_t device, const float* sum_f32, size_t n_elems, void* out_bf16, void* cuda_stream);

/* End-to-end convenience: same as slp_moe_prefill but hidden/out are HOST buffers ([T,H] bf16,
 * pinned for full speed); copies in and out through an internal device buffer on the internal
 * compute stream and returns when `out` is complete. */
slp_status slp_moe_prefill_host(slp_moe_layer* h, const void* hidden_bf16_host, int32_t T, void* out_bf16_host);

/* Waits for the in-flight call (if any) and releases everything create allocated or pinned. */
slp_status slp_moe_layer_destroy(slp_moe_layer* h);

/* Thread-local description of the last error on this thread ("" if none). */
const char* slp_last_error(void);

/* Parity / evidence exports.  Each waits for the in-flight call, then copies device -> host. */
slp_status slp_moe_debug_routing(slp_moe_layer* h, int32_t* idx /*[T,k]*/, float* w /*[T,k]*/, int32_t* counts /*[E]*/);
slp_status slp_moe_debug_quant_hidden(slp_moe_layer* h, uint8_t* xq /*[T,H]*/, float* xs /*[T,H/128]*/);
/* Copies min(bytes, size of the buffer for the last call) bytes; *written gets that size. */
slp_status slp_moe_debug_buffer(slp_moe_layer* h, int32_t which, void* host_dst, size_t bytes, size_t* written);
/* Copies `bytes` bytes starting `offset` bytes into the same buffer (full-size parity tests read single
 * experts' rows of hq / hs / Y instead of gigabytes).  INVALID_ARG if the range leaves the buffer. */
slp_status slp_moe_debug_buffer_range(slp_moe_layer* h, int32_t which, size_t offset, size_t bytes, void* host_dst);
slp_status slp_moe_get_stats(slp_moe_layer* h, slp_moe_stats* stats);

/* Bring-up / bisection only, not a product option: the NEXT slp_moe_layer_create / slp_moe_stack_create on the calling
 * thread builds its handle with the kernel variants or the workspace canary bands `spec` names (comma-separated:
 * "gemm=simt", "gemm=static", "gemm=pair", "router=fp32", "guards", "guards=selftest"), then the setting is
 * gone.  NULL or "" = the product path (and cancels a pending setting).  Thread-local: creates on other threads are
 * not affected, and the library reads no environment variable.  INVALID_ARG for an unknown token. */
slp_status slp_moe_debug_set_triage(const char* spec);

/* Measures pinned host -> device bandwidth on `device` with back-to-back cudaMemcpyAsync of
 * `chunk_bytes` each (total `total_bytes`, best of `repeats`); writes GB/s (1e9) to *gbs.
 * This is the denominator of the streamed-mode roofline. */
slp_status slp_measure_h2d(int32_t device, size_t chunk_bytes, size_t total_bytes, int32_t repeats, double* gbs);

/* The histogram / scan / permute step (Fig. 2 step 4: tokens "sorted to form per-expert token lists") as a
 * stand-alone call that NEVER allocates: no handle, no cudaMalloc / cudaFree / cudaMallocHost, no allocating
 * library routine, on the first call or any later one.
 *
 * It exists for callers that cannot obtain device memory at the point where they need this step: a serving process whose
 * own pool allocator took all of HBM at start-up (a cudaMalloc would fail, or steal from the pool's accounting); a
 * plugin invoked inside a region where its host forbids driver allocations because they synchronise the device
 * (latency-critical decode loops); code running after the device is already full.  The handle-based calls above
 * cannot serve them, because slp_moe_layer_create allocates.  Here the caller brings every input and output buffer and
 * the step's scratch (per-chunk expert histograms and the tile tables the scan emits) lives in one 616 KiB array
 * compiled into the library.  Cost: each GPU on which the process uses this library holds those 616 KiB from the moment
 * the library is loaded there until the process exits, whether or not this function is ever called.
 *
 * Limits (SLP_ERR_UNSUPPORTED_SHAPE beyond them, nothing launched): T <= 32768 tokens, T * top_k <= 262144 routed
 * assignments, 1 <= n_experts <= 511, 1 <= top_k <= min(32, n_experts).  T == 0 returns SLP_OK and touches nothing.
 *
 *  idx_dev        dev [T, top_k] int32, read only: the experts of each token, every entry in [0, n_experts)
 *                 (an entry outside that range is undefined behaviour, as in slp_moe_prefill's own router output).
 *  counts_dev     dev [n_experts] int32, out: tokens per expert.
 *  row_start_dev  dev [n_experts + 2] int32, out: first workspace row of each expert's 128-aligned range; entry
 *                 n_experts = 0 (the un-permuted rows [0, T) in front, the shared expert's rows); entry
 *                 n_experts + 1 = rows in use.
 *  pos_dev        dev [T, top_k] int32, out: workspace row of assignment (t, j); rows of one expert ascend with t.
 *  row_token_dev  dev [row_capacity] int32, out: token of each workspace row, -1 in padding rows.  The first
 *                 slp_moe_permute_static_rows(T, top_k, n_experts) entries are overwritten, later ones untouched.
 *  row_capacity   entries row_token_dev can hold; must be >= slp_moe_permute_static_rows(...) (the data-independent
 *                 worst case; INVALID_ARG otherwise).
 *  cuda_stream    a cudaStream_t on `device`; the call is asynchronous on it like slp_moe_prefill.
 * The layouts are those of SLP_BUF_COUNTS / ROW_START / POS / ROW_TOKEN of an unsharded handle, bit for bit.
 *
 * First call on a device: the function looks up where that device's copy of the scratch array lives (one
 * cudaGetSymbolAddress, with `device` made current, result cached per device under a mutex).  That is a set-up step;
 * make the first call on each device outside any stream capture.  The function makes `device` current and leaves it so.
 *
 * One array per device, shared by every call from every thread and stream: two calls on the same device whose kernels
 * can overlap on the GPU (different streams without an event between them) race on it and both results are garbage.
 * Order them on one stream or with events.  The array keeps the previous call's contents; the call itself
 * re-initialises everything it reads, so no clearing is needed between calls. */
slp_status slp_moe_permute_static(int32_t device, const int32_t* idx_dev, int32_t T, int32_t top_k, int32_t n_experts,
                                  int32_t* counts_dev, int32_t* row_start_dev, int32_t* pos_dev, int32_t* row_token_dev,
                                  int64_t row_capacity, void* cuda_stream);

/* Host arithmetic only: the number of int32 entries slp_moe_permute_static needs in row_token_dev,
 * roundup128(T) + roundup128(T * top_k + 127 * n_experts); -1 for a negative argument. */
int64_t slp_moe_permute_static_rows(int32_t T, int32_t top_k, int32_t n_experts);

/* Library version string, "slpmoe <release> (sm_100a; abi <SLP_MOE_ABI_VERSION>)". */
const char* slp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SLP_MOE_H */
