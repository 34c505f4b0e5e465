/*
 * af.h — C ABI of the B200-native Cross-Request State Packed Forward over a Unified KV Ring Buffer
 * (ActionFlow, arxiv 2512.20276).  Citations "P:<n>" are lines of /root/reference/PAPER.md.
 *
 * What the library computes
 *   One call of af_packed_forward is Algorithm 2 "Cross-Request State Packed Forward" applied
 *   for every layer l = 0..n_layers-1 (Alg. 1 line 3 "PackedForwardEachLayer") to the packed
 *   Cross-Request State H_CRS of Eq. 1: the rows of all segments (one prefill segment of L_P rows
 *   and K-1 single-row decode segments in the paper's schedule) stacked along the sequence dimension.
 *   Per layer: RMSNorm -> QKV projection -> RoPE at the token's logical position in its own request and append
 *   of K/V into the Unified KV Ring Buffer -> segment-wise causal attention, every row
 *   attending to positions 0..own position of its own request only -> output projection + residual
 *   -> RMSNorm -> SwiGLU MLP + residual (P:185 read as the standard Llama pre-norm block, reading A1).
 *   af_logits_rows is LMHead(Norm(H[s])) of Alg. 1 lines 5/8 on a caller-chosen row list.
 *   The paper's InPlaceShiftKV moves no bytes here: regions are keyed by req_id and the stage
 *   shift is a relabelling (reading A7); af_ring_reset_slot recycles an evicted request's region.
 *
 * Conventions
 *   - All "device" pointers are CUDA device memory of the current device, owned by the caller.
 *     All "host" pointers are ordinary host memory, read (or written) before the call returns.
 *   - bf16 = bfloat16, fp16 = IEEE binary16, both stored as uint16.  Weights, gains and the packed embeddings are bf16;
 *     weights are [out_features, in_features] row-major (y = x W^T).  The KV ring holds fp16 (same bytes as bf16, 3 more
 *     mantissa bits: DESIGN.md "Precision"); all accumulation and the residual stream are fp32.
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t cast to void*) and return without host synchronisation
 *     (the af_debug_* calls of af_debug.h synchronise; they are test/bench helpers, not the hot path).
 *   - Devices and streams.  The library keeps nothing process-global that kernels synchronise through: its schedule
 *     tables are per device, its stream-K flags and the layer-chain kernel's grid barrier per (device, stream).  Its
 *     persistent kernels wait inside themselves (stream-K owners for contributors of their own launch, the chain for its
 *     own grid barrier), so they need their whole grid resident: grids are sized with the occupancy API for the current
 *     device, and a step enqueued on one stream is ordered (cudaStreamWaitEvent) behind the library work last enqueued on
 *     another stream of the same device - two rings driven from two streams are correct, but never overlap.  Other
 *     work of the caller that occupies SMs while a step runs only delays it (a stream-K owner waits for CTAs dispatched
 *     before it, never after); it must not itself wait for the step.  Every such wait is bounded: a CTA that waits ~4 s
 *     for another CTA of its grid traps, and the stream reports a launch failure (AF_ERR_CUDA on the next call) instead
 *     of hanging the device.
 *   - fp16 range.  Values stored as fp16 (q, k, v, attention output, the SwiGLU product, the partial sums exchanged
 *     between CTAs) are converted with saturation: a finite value beyond +-65504 becomes +-65504, never inf.
 *   - Return value: 0 on success, a negative AF_ERR_* otherwise.  On any error raised by argument validation
 *     no kernel has been launched and the ring bookkeeping is unchanged.  af_last_error() gives a message.
 *   - One af_ring is not thread-safe; the caller serialises calls on it (different rings may be driven from different
 *     host threads and streams).
 *   - There is no CPU fallback anywhere in this library.
 *
 * Ring geometry (reading A6).  One allocation `kv_mem` holds, for every layer, all R = n_regions
 *   request regions of C = capacity token slots each ("single, circular, physically contiguous memory region ...
 *   logically partitioned per request").  The token at logical position pos of request r lives in
 *       slot      = (base_r + pos) mod C                       (slot inside region r)
 *       row_slot  = r * C + slot                               (the global slot id reported by af_debug_row_map)
 *   and its K (after RoPE) and V vectors of head h are the head_dim contiguous fp16 values at element offset
 *       (((layer * 2 + kv) * R + r) * n_heads + h) * C * head_dim + slot * head_dim,     kv = 0 for K, 1 for V.
 *   A request's live range is positions 0..len_r-1; slots outside it are never read.
 */
#ifndef AF_H_
#define AF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AF_OK               0
#define AF_ERR_ARG         (-1)  /* null pointer, non-positive size, misaligned pointer */
#define AF_ERR_SEGMENT     (-2)  /* bad or duplicate req_id, len < 1, decode segment with len != 1, too many segments */
#define AF_ERR_POSITION    (-3)  /* start_pos != current length of the request (appends must be contiguous) */
#define AF_ERR_CAPACITY    (-4)  /* start_pos + len > capacity: a live token would be overwritten */
#define AF_ERR_WORKSPACE   (-5)  /* workspace / kv_mem too small */
#define AF_ERR_CUDA        (-6)  /* a CUDA runtime/driver call failed */
#define AF_ERR_UNSUPPORTED (-7)  /* shape outside what the sm_100a kernels handle */

#define AF_PHASE_PREFILL 0
#define AF_PHASE_DECODE  1
#define AF_MAX_SEGS      64      /* segments per packed step */

typedef struct af_ring af_ring;  /* opaque, library-owned */

typedef struct {
  int32_t d_model, n_layers, n_heads, head_dim, ffn, vocab;  /* d_model == n_heads*head_dim; head_dim in {64,128} */
  float   rms_eps, rope_theta;
} af_model_cfg;

typedef struct { int32_t n_regions, capacity; } af_ring_cfg;

/* One segment of the packed step = "append len tokens at positions start_pos..start_pos+len-1 of request req_id"
 * (the segment lengths L_s of Alg. 2).  Rows of packed_embeds follow the segment-table order. */
typedef struct { int32_t req_id, phase, start_pos, len; } af_segment;

typedef struct {                 /* all device bf16 */
  const void *wq, *wk, *wv, *wo; /* [d_model, d_model] */
  const void *w_gate, *w_up;     /* [ffn, d_model] */
  const void *w_down;            /* [d_model, ffn] */
  const void *g_attn, *g_mlp;    /* RMSNorm gains [d_model] */
} af_layer_weights;

#define AF_WEIGHTS_BF16 0         /* projection matrices are bf16; every weight tile is converted to fp16 in shared memory */
#define AF_WEIGHTS_FP16 1         /* projection matrices were prepared once with af_convert_bf16_to_fp16 (same values) */
#define AF_WEIGHTS_FP16_GU 2      /* as AF_WEIGHTS_FP16, and w_gate of every layer holds gate AND up, interleaved by
                                   * af_prepare_gate_up (w_up is ignored): one TMA box per weight tile instead of eight */

#define AF_WEIGHTS_FP8 3          /* f4, weight-only FP8 storage: wq..w_down hold one E4M3 code per element
                                   * (uint8, [out, in] row-major), w_gate holds gate AND up interleaved by
                                   * af_prepare_gate_up_fp8 (w_up is ignored), af_weights.scales holds one fp32 scale per
                                   * OUTPUT channel; the matrix the library multiplies by is value(code) * scale[out].
                                   * The codes are widened to fp16 (exactly) tile by tile in shared memory and the scale
                                   * is applied to the fp32 accumulator, so HBM carries half the bytes of the 16-bit
                                   * formats.  w_lm stays a prepared fp16 matrix.  Packed steps of more than 1024 rows
                                   * return AF_ERR_UNSUPPORTED in this format. */

typedef struct {                  /* AF_WEIGHTS_FP8: device fp32 [out_features] per matrix */
  const float *sq, *sk, *sv, *so; /* [d_model] */
  const float *s_gate, *s_up;     /* [ffn] */
  const float *s_down;            /* [d_model] */
} af_layer_scales;

typedef struct {
  af_model_cfg cfg;
  const af_layer_weights* layers; /* HOST array [n_layers] of device pointers */
  const void* g_final;            /* device bf16 [d_model] */
  const void* w_lm;               /* device bf16 (or prepared fp16) [vocab, d_model] */
  int32_t weight_format;          /* AF_WEIGHTS_BF16, _FP16, _FP16_GU or _FP8: format of wq..w_down (and, except for _FP8, of w_lm); gains stay bf16 */
  const af_layer_scales* scales;  /* HOST array [n_layers] of device pointers; read only when weight_format == AF_WEIGHTS_FP8 */
} af_weights;

/* Load-time weight preparation: dst[i] = fp16(src[i]) for n_elems bf16 values (n_elems % 8 == 0,
 * both device, 16-byte aligned, may not overlap).  Exact for every finite bf16 value with 2^-14 <= |w| <= 65504; smaller
 * values round to fp16 subnormals (absolute error <= 2^-25).  Enqueued on cuda_stream. */
int af_convert_bf16_to_fp16(const void* src_bf16, void* dst_fp16, size_t n_elems, void* cuda_stream);

/* Load-time preparation of the MLP input projections for AF_WEIGHTS_FP16_GU: converts gate and up ([ffn, d_model]
 * bf16, device) to fp16 like af_convert_bf16_to_fp16 and writes them as ONE matrix dst_fp16 of
 * af_gate_up_rows(ffn) x d_model in the row order the SwiGLU epilogue wants (h = silu(gate) * up): for
 * every tile t of 64 features and every quarter q of it, 16 gate rows (features 64t + 16q ..) followed by the 16 up
 * rows of the same features; rows of features >= ffn are zero.  dst_fp16 is caller-owned (device, 16-byte aligned,
 * d_model % 8 == 0).  Enqueued on cuda_stream. */
size_t af_gate_up_rows(int32_t ffn);
int af_prepare_gate_up(const void* gate_bf16, const void* up_bf16, void* dst_fp16, int32_t ffn, int32_t d_model,
                       void* cuda_stream);

/* AF_WEIGHTS_FP8: the same row order for E4M3 codes (one byte per element; copied, not converted).  gate / up are
 * [ffn, d_model] uint8, dst is af_gate_up_rows(ffn) x d_model uint8, rows of features >= ffn are zero codes; all device,
 * 16-byte aligned, d_model % 16 == 0.  Enqueued on cuda_stream. */
int af_prepare_gate_up_fp8(const void* gate_codes, const void* up_codes, void* dst_codes, int32_t ffn, int32_t d_model,
                           void* cuda_stream);

/* Bytes of kv_mem needed for (cfg, ring): 2 * n_layers * R * n_heads * C * head_dim * 2. */
size_t af_ring_bytes(const af_model_cfg* cfg, const af_ring_cfg* ring);
/* Bytes of workspace needed by af_packed_forward / af_logits_rows for up to max_rows packed rows. */
size_t af_workspace_bytes(const af_model_cfg* cfg, int32_t max_rows, int32_t max_segs);

/* Create the ring bookkeeping over caller-owned device memory kv_mem (256-byte aligned, >= af_ring_bytes).
 * All regions start with base = 0, len = 0.  kv_mem is not touched (stale bytes are unreachable).
 * The library allocates only small device metadata of its own (RoPE table, segment tables). */
int af_ring_create(const af_model_cfg* cfg, const af_ring_cfg* ring, void* kv_mem, size_t kv_bytes, af_ring** out);

/* Recycle region req_id for a new request ("overwriting the evicted oldest request", with no copy):
 * len = 0 and base = new_base mod C if new_base >= 0, else base = (base + len) mod C (keep rotating). O(1), host only. */
int af_ring_reset_slot(af_ring* ring, int32_t req_id, int32_t new_base);

/* f3 - sliding window inside a request ("updates the ring buffer's sliding window, discarding stale tokens";
 * DESIGN.md A8b).  window = 0 (the default after af_ring_create) keeps the v1 rule start_pos + len <= capacity.  With
 * 1 <= window <= capacity a request may grow up to max_pos (>= capacity; 0 = capacity) tokens: the append at position p
 * goes to slot (base + p) mod C and overwrites position p - C, and the row at position p attends positions
 * max(0, p - window + 1)..p of its request only.  All rows of a step are appended before any row attends, so a segment
 * that ends beyond capacity needs len <= capacity - window + 1 (AF_ERR_CAPACITY otherwise, state unchanged).  Every
 * region must be empty (AF_ERR_POSITION otherwise).  Rebuilds the library's RoPE table for max_pos positions;
 * synchronises, not hot path. */
int af_ring_set_window(af_ring* ring, int32_t window, int32_t max_pos);

/* Algorithm 2 for all layers on one packed step.
 *   packed_embeds : device bf16 [T, d_model], T = sum of segment lens, rows in segment-table order (H_CRS, Eq. 1)
 *   segs          : HOST array [n_segs]; each req_id at most once; start_pos == current len of that request;
 *                   start_pos + len <= capacity (unless af_ring_set_window relaxed it); phase == AF_PHASE_DECODE
 *                   requires len == 1.  n_segs == 0 is a no-op.
 *   hidden_out    : device fp32 [T, d_model], the residual stream after the last layer (before the final norm)
 *   workspace     : device, 256-byte aligned, >= af_workspace_bytes(cfg, T, n_segs)
 * On success the ring lengths advance: len_r = start_pos + len for every segment (the "ring commit"). */
int af_packed_forward(const af_weights* w, const void* packed_embeds, const af_segment* segs, int32_t n_segs,
                      af_ring* ring, float* hidden_out, void* workspace, size_t ws_bytes, void* cuda_stream);

/* logits_out[i, :] = RMSNorm(hidden[rows[i], :]; g_final) W_lm^T   (Alg. 1 l.5/l.8).
 *   hidden : device fp32 [>= max(rows)+1, d_model];  rows : HOST int32 [n_rows], n_rows <= 256
 *   logits_out : device fp32 [n_rows, vocab] */
int af_logits_rows(const af_weights* w, const float* hidden, const int32_t* rows, int32_t n_rows,
                   float* logits_out, void* workspace, size_t ws_bytes, void* cuda_stream);

/* ---- the device half of Alg. 1's loop around the forward ----
 * tokens_out[i] = ArgMax_v logits[i, v]  (Alg. 1 l.5 / l.8 "ArgMax(LMHead(Norm(H[s])))").  Ties go to the LOWEST index;
 * NaN entries are never selected (a row of only NaNs gives 0).  An integer decided by floating point: it is taken on
 * the fp32 logits exactly as stored, so any implementation given the same logits returns the same tokens.
 *   logits : device fp32 [n_rows, vocab] (row pitch = vocab);  tokens_out : device int32 [n_rows].  Enqueued. */
int af_argmax_rows(const float* logits, int32_t n_rows, int32_t vocab, int32_t* tokens_out, void* cuda_stream);

/* af_argmax_rows for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same result (the rule above is order-free, so the tokens are identical), no
 * cudaMalloc / cudaFree / allocating library routine on any call, the first included.  Every row's vocabulary is split
 * over up to 64 CTAs; their candidates and one arrival counter per row live in a static __device__ array inside the
 * library (131 KB of device memory that every GPU which loads the library holds until exit).
 *   n_rows <= AF_ARGMAX_STATIC_MAX_ROWS, else AF_ERR_UNSUPPORTED (nothing enqueued; use af_argmax_rows).
 *   Every call on a device shares that array, which keeps the last call's contents; the call clears the counters it
 *   uses (a memset enqueued before the kernel).  Calls that OVERLAP on the GPU (two streams, or two processes' worth of
 *   threads on one device) race on it and return wrong tokens: order them on one stream or with events.  Enqueued. */
#define AF_ARGMAX_STATIC_MAX_ROWS 256
int af_argmax_rows_static(const float* logits, int32_t n_rows, int32_t vocab, int32_t* tokens_out, void* cuda_stream);

/* embeds_out[i, :] = table[tokens[i], :]  (the token half of Alg. 1 l.2 "Embed(.., GetLastTokenEach(A_sequences))",
 * P:134): the rows a step's decode segments take as input.  A copy, bit-exact.
 *   table : device bf16 [vocab, d_model] (d_model % 8 == 0, 16-byte aligned);  tokens : device int32 [n_rows], each in
 *   [0, vocab) (a token outside the range writes a row of zeros);  embeds_out : device bf16 [n_rows, d_model],
 *   typically rows of the next step's packed_embeds.  Enqueued. */
int af_embed_rows(const void* table, int32_t vocab, int32_t d_model, const int32_t* tokens, int32_t n_rows,
                  void* embeds_out, void* cuda_stream);

/* ---- f1, second half: Algorithm 1's pipeline loop with its state on the device ----
 * An af_loop drives the paper's K-stage pipeline over one ring: step t packs the prefill of frame t (prefill_len rows,
 * region t mod R, recycled first exactly as af_ring_reset_slot(ring, t mod R, -1)) with decode stage s = 1..min(t, K-1)
 * of frame t-s (region (t-s) mod R, position prefill_len + s - 1; Alg. 1 l.2-10).  The segment table,
 * the per-region (base, len) bookkeeping and A_sequences live in device memory and are advanced by kernels; the decode
 * rows are Embed(ArgMax(logits of the previous step)) (af_embed_rows / af_argmax_rows' kernels, lowest index wins).
 * The host keeps an integer mirror (the ring's own) for validation and launch geometry only.  Once the pipeline is
 * full every step has the same shape: the first full step is issued as plain launches, the second is captured into
 * ONE CUDA graph, later steps replay it (use_graph != 0 and a non-default stream; otherwise plain launches).  No call
 * synchronises.
 *   af_loop_create : w (needs g_final, w_lm; the struct is copied, w->layers must outlive the loop), ring (all regions
 *     are emptied at their current rotation; the loop owns the ring's bookkeeping until af_loop_destroy), embed_table =
 *     device bf16 [vocab, d_model], 16-byte aligned, caller-owned; workspace as for af_packed_forward with
 *     max_rows >= prefill_len + chunk_k - 1, caller-owned, must outlive the loop.  Needs chunk_k <= n_regions
 *     (AF_ERR_SEGMENT) and prefill_len + chunk_k - 1 <= capacity (AF_ERR_CAPACITY).  The loop's own buffers (a few MB)
 *     are library-owned device memory.
 *   af_loop_buffers : device pointers, each may be NULL: prefill_embeds = bf16 [prefill_len, d_model], the caller writes
 *     frame t's projected embeddings here on `cuda_stream` before af_loop_step; hidden = fp32 [T, d_model] and
 *     logits = fp32 [1 + n_dec, vocab] of the last step (prediction rows in stage order); tokens = int32 [1 + n_dec]
 *     tokens of the last step by stage; frame = int32 [1 + chunk_k]: {frame id, its chunk_k tokens} of the last
 *     COMPLETED frame (id -1 while the pipeline fills).
 *   af_loop_step : enqueues step t on cuda_stream and advances the host mirror.  If a launch fails (AF_ERR_CUDA) the
 *     loop and its ring are left in an unspecified state and must be destroyed.
 *   af_loop_steps_done : t, the number of steps enqueued so far (-1 for a NULL loop). */
typedef struct af_loop af_loop;
int af_loop_create(const af_weights* w, af_ring* ring, const void* embed_table, int32_t prefill_len, int32_t chunk_k,
                   void* workspace, size_t ws_bytes, af_loop** out);
int af_loop_buffers(af_loop* loop, void** prefill_embeds, float** hidden, float** logits, int32_t** tokens, int32_t** frame);
int af_loop_step(af_loop* loop, int32_t use_graph, void* cuda_stream);
int32_t af_loop_steps_done(const af_loop* loop);
int af_loop_destroy(af_loop* loop);

int af_ring_destroy(af_ring* ring); /* frees the handle and its own metadata; never frees caller memory */

/* Introspection (row map, bookkeeping), per-kernel timing, the GEMM work lists and the chain kernel's timeline are test /
 * bench helpers, not the product path: they are declared in include/af_debug.h (same library). */

const char* af_last_error(void); /* thread-local message of the last failing call */

#ifdef __cplusplus
}
#endif
#endif /* AF_H_ */
