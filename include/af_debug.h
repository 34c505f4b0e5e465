/*
 * af_debug.h - test / bench helpers of libaf_b200.so (introspection, per-kernel timing, GEMM work lists, the layer-chain
 * kernel's timeline).  Not the product path: these calls synchronise the device.  See include/af.h for the C ABI proper.
 */
#ifndef AF_DEBUG_H_
#define AF_DEBUG_H_

#include "af.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ---- introspection for bit-exact bookkeeping parity; these synchronise, they are not hot path ---- */
int af_ring_get_state(const af_ring* ring, int32_t req_id, int32_t* base, int32_t* len);
/* Row map of the LAST af_packed_forward, copied back from the DEVICE tables the kernels used.
 * Each output is a HOST int32 [n] array (n <= T of that step) or NULL. */
int af_debug_row_map(const af_ring* ring, int32_t* row_req, int32_t* row_pos, int32_t* row_slot, int32_t n);
/* Bench/test only: rewind (or set) the bookkeeping length of a region; moves no data. */
int af_debug_set_len(af_ring* ring, int32_t req_id, int32_t len);
/* Number of kernel launches issued by this library since load (for bench.py's gpu_launches). */
int64_t af_debug_launch_count(void);
/* Plain C = A B^T through the same tcgen05 GEMM kernel the forward uses (unit tests / roofline probes).
 * a: device fp16 [n_tok, k] (activations), w: device bf16 [n_out, k]; out: device fp32 [n_tok, n_out], n_out % 4 == 0. */
int af_debug_gemm(const void* a, const void* w, float* out, int32_t n_tok, int32_t n_out, int32_t k,
                  void* workspace, size_t ws_bytes, void* cuda_stream);

/* Per-kernel-class timing with CUDA events on the launching stream (bench.py's roofline leg; adds event records
 * between kernels, so it is switched on only for a separate profiling pass).  Classes, in order: gemm_qkv, gemm_o,
 * gemm_gateup, gemm_down, gemm_lm, attention, rope_append, rmsnorm, chain (layer_chain_kernel launches), other (10 slots).
 * enable = 1: time the path as it runs; enable = 2: also force the per-stage path (one kernel per stage) instead of the
 * layer chain, so that every stage has a class of its own; 0: off.
 * af_debug_profile_read synchronises, returns summed milliseconds and launch counts since the last read, and clears. */
int af_debug_profile(int enable);
/* Which kernel runs the attention stage (a4).  The units of attention_umma.cuh (tensor units on tcgen05 for multi-row
 * segments, row units for one-row segments; head_dim 128, no window, every segment's context <= 352) run as the last phase
 * of the layer chain, or as attention_umma_kernel on the per-stage path; attention_kernel (mma.sync; any head_dim, window,
 * context) is a kernel of its own.  mode 0 (default): the units for steps made of one-row segments only (decode-only
 * steps, where they are 2-4 % faster per step), attention_kernel for every other step (1.5 % faster there).
 * mode 1: attention_kernel always.  mode 2: the units wherever they apply.  Process-wide; takes effect at the next
 * af_packed_forward / captured graph. */
int af_debug_attention(int mode);
int af_debug_profile_read(double* ms_sum, int64_t* counts, int32_t n_slots);

/* The work lists of the GEMM kernel (pure host logic, needs no GPU): for `n_tile_pairs` pairs of 128-row weight tiles and
 * `n_kblocks` 64-wide k-blocks on at most `max_clusters` 2-CTA clusters: stream-K ranges (split_k == 0), split-K (split_k ==
 * 1: `splits` equal slabs per tile pair) or the layer chain's slab ranges (split_k == 2: equal unit ranges, every piece a
 * plain piece stored as slab `slab` = its ordinal inside its tile pair, at most `splits` per pair) or the skewed split-K of a
 * launch's first phase (split_k == 3: clusters numbered split-major, k-ranges shrinking from the first split to the last).  pieces = HOST int32 [max_clusters_out][16][8]; piece = {pair, kb0, kb1, kind (0 plain,
 * 1 contributor, 2 owner), slot, n_contrib, slab, 0}, a cluster's list ends at pair = -1.  Returns the number of
 * clusters used, or a negative AF_ERR_*. */
int af_debug_gemm_schedule(int32_t split_k, int32_t n_tile_pairs, int32_t n_kblocks, int32_t max_clusters, int32_t splits,
                           int32_t* pieces, int32_t max_clusters_out);

/* Debug timeline of the layer-chain kernel: while enabled every layer_chain_kernel launch records %globaltimer stamps per
 * CTA (slot 0: start, after griddepcontrol.wait; slot 1 + 2p: phase p's work done; slot 2 + 2p: the grid barrier after
 * phase p passed) into a library-owned device buffer that keeps the last 16 launches.  af_debug_trace_read synchronises
 * and copies them out: stamps = HOST int64 [16][160][18], meta = HOST int32 [16][2] (phases of the launch, grid size);
 * returns the number of launches recorded since af_debug_trace(1), or a negative AF_ERR_*. */
int af_debug_trace(int enable);
int af_debug_trace_read(long long* stamps, int* meta);

#ifdef __cplusplus
}
#endif
#endif /* AF_DEBUG_H_ */
