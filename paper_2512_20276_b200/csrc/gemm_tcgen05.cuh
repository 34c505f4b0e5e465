// Packed-projection GEMM for sm_100a: out[token, feature] (op)= sum_k X[token, k] * W[feature, k]
// (steps a2/a5/a7/a8/a10 of SURVEY.md 8(a); Alg. 2 lines 2 and 6).  DESIGN.md section 6.1.
//
// "Swap-AB" orientation: the WEIGHT tile (128 output features x 64 k) is the UMMA A operand and the packed TOKEN tile
// (all T <= 512 tokens x 64 k of a launch) is the B operand, so the 282-row packed matrix of the paper's schedule maps onto UMMA
// N = 2 x 144 with 2% padding instead of 3 x 128-row M tiles with 27% padding, and a decode-only step (T <= 16) uses
// N = 16.  Both operands are K-major in global memory, are staged by TMA with the 128-byte swizzle, and are consumed by
// tcgen05.mma kind::f16 (fp16 activations x fp16 weights - prepared at load time, or bf16 weights rewritten as fp16 per
// tile in shared memory - with the fp32 accumulator in TMEM).
//
// The grid is launched in 2-CTA clusters whose work unit is (pair of neighbouring weight tiles, k-block):
//   kMma2 = true   the pair's leader issues tcgen05.mma.cta_group::2 (M = 256); each CTA stages its weight tile and
//                  half of the activation rows (34 KB per stage at T = 282); the peer's loads complete on the leader's
//                  mbarrier and the leader's commits are multicast to both CTAs.
//   kMma2 = false  cta_group::1 MMAs per CTA; the activation boxes are TMA-multicast across the cluster.
//
// Work split over a persistent grid (<= 1 CTA per SM), two modes:
//   SPLIT_STREAMK  contiguous ranges of units per cluster.  A CTA that holds a k-tail of a tile (always the FIRST
//                  piece of its range) writes its partial (fp16 in the forward, fp32 in af_debug_gemm) to the workspace
//                  and raises a flag; the CTA that holds the k-head (always the LAST piece of its range, so the
//                  partials were written long before) pulls them into the freed pipeline stages with bulk copies,
//                  adds them in CTA order (deterministic) and runs the epilogue.
//   SPLIT_K        every tile is cut into `splits` equal k-ranges, one CTA each; every CTA stores its partial slab
//                  [split][token][feature] and the NEXT kernel (residual + RMSNorm, elementwise.cuh) adds the slabs in
//                  split order.  No CTA ever waits on another.
//
// Epilogues (features sit on TMEM lanes, tokens on columns), per warp and 32-token chunk.  The drain is bound by the
// TMEM read port (64 B/clk per SM: 128 lanes x 288 fp32 columns = 2300 clk), so everything else is kept off its path:
//   fp16 outputs   (every GEMM of the forward; kernel variant kFrag) tcgen05.ld.16x256b delivers the accumulator in
//                  the mma fragment layout (thread t: feature t/4 [+8], tokens 2(t%4), +1 of every 8), which four
//                  stmatrix.trans write as a swizzled [token][feature] image in the warp's 2 KB staging buffer; the
//                  warp reads the image back row-wise and stores 16 bytes per lane to global memory (64 contiguous
//                  bytes per token).  The TMEM load of the next chunk is in flight meanwhile.  No TMA store, no
//                  proxy fence, no bulk-group wait.  Stream-K partials are the same images written raw (2 KB each)
//                  and are added by the owner with ldmatrix.trans in the same layout.
//   fp32 outputs   (LM head, af_debug_gemm) tcgen05.ld.32x32b, one feature per lane, staged [token][feature] in
//                  shared memory and written with TMA tensor stores; fp32 partials likewise through map_part.
//   EPI_STORE      plain store (q|k|v, split-K slabs, logits).
//   EPI_SWIGLU     tile = 64 gate rows + 64 up rows of the same features, loaded so that every lane quadrant holds
//                  16 gate + 16 up rows of the same 16 features: in the fragment layout gate and up of one (feature,
//                  token) sit in the same thread (registers j and 16 + j); the output is fp16(silu(gate) * up).
//
// Warp roles (320 threads): warps 0-7 epilogue (TMEM lane quadrant = warp % 4, two warps per quadrant alternate
// 32-token chunks; with bf16 weights they also run the per-tile weight transform), warp 8 TMA producer, warp 9 MMA issuer.
#pragma once
#include "ptx.cuh"

// epilogue warps: 8, 12 or 16 (-DAF_EPI_WARPS=...); 12 and 16 were measured on B200 and are no faster than 8
#ifndef AF_EPI_WARPS
#define AF_EPI_WARPS 8
#endif
#if AF_EPI_WARPS == 8
#define AF_EPI_THREADS 256
#elif AF_EPI_WARPS == 12
#define AF_EPI_THREADS 384
#elif AF_EPI_WARPS == 16
#define AF_EPI_THREADS 512
#endif

namespace af {

constexpr int GEMM_BM = 128;       // weight rows (output features) per tile = UMMA M
constexpr int GEMM_BK = 64;        // bf16 elements per k-block = one 128-byte swizzle row
constexpr int GEMM_EPI_WARPS = AF_EPI_WARPS;  // two per TMEM lane quadrant (warp % 4), alternating 32-token chunks
constexpr int GEMM_THREADS = (GEMM_EPI_WARPS + 2) * 32;
constexpr int GEMM_BLK = 32 * (GEMM_EPI_WARPS / 4);  // columns one round of the epilogue warps covers
constexpr int GEMM_MAX_TOK = 512;  // tokens per launch: one UMMA N <= 256, or two halves of <= 256 (all 512 TMEM columns)
constexpr int GEMM_TMEM_COLS = 512;
constexpr int GEMM_MAX_STAGES = 12;
constexpr int GEMM_XCH_MAX = GEMM_EPI_WARPS * 8192;  // per epilogue warp: two 4 KB (or one 2 KB) staging buffers for TMA stores
constexpr int GEMM_SMEM_BUDGET = 232448 - 1024 - 2304;   // dynamic shared memory: 227 KB minus the static part (layer_chain_kernel: + AuLists)

enum GemmEpilogue : int { EPI_STORE = 0, EPI_SWIGLU = 1 };
enum GemmSplit : int { SPLIT_STREAMK = 0, SPLIT_K = 1 };

// One piece of a cluster's work: k-blocks [kb0, kb1) of tile pair `pair` (CTA r of the cluster computes tile
// pair * cluster + r).  PK_PLAIN pieces cover a whole tile (or, in SPLIT_K mode, one slab `mid` of it) and are
// drained straight to the output; a PK_CONTRIB piece writes its partial to slot `slot` and raises the slot's flag;
// a PK_OWNER piece waits for the n_contrib partials in slots [slot, slot + n_contrib), adds them (in slot order) to
// its own accumulator (nothing of its own when kb0 == kb1) and runs the epilogue.  The host builds the lists so that
// contributor pieces come first in their cluster and owner pieces last (af_lib.cu, build_schedule).
enum GemmPieceKind : int { PK_PLAIN = 0, PK_CONTRIB = 1, PK_OWNER = 2 };
struct alignas(16) GemmPiece { int pair, kb0, kb1, kind, slot, n_contrib, mid, pad; };
constexpr int GEMM_MAX_PIECES = 16;

// The output is written with TMA tensor stores through map_out, a rank-3 view (feature, middle, token) of the
// destination: middle = weight part (q|k|v stacked along the feature axis) or split-K slab; the map's extents clip
// ragged feature tiles and the token padding.
struct GemmParams {
  int n_parts;         // weight matrices stacked along the feature axis (q|k|v): 1..3 (when a_pair == 0)
  int part_rows;       // output features per part (a_pair: rows of gate = rows of up)
  int tiles_per_part;  // ceil(part_rows / 128)
  int a_pair;          // 2: map_w0 holds gate | up interleaved at load time (af_prepare_gate_up), tile t = its rows [128t, +128);
                       // 1: tile t = rows [64t, 64t+64) of map_w0 (gate) and of map_w1 (up), interleaved 16 + 16 per lane quadrant
  int K, num_kb;       // reduction length, ceil(K / 64)
  int T, tok0;         // valid tokens of this launch, first token row
  int n1, n2;          // UMMA N of the two token halves (multiples of 16, n2 may be 0)
  int xh;              // token rows per activation TMA box (two boxes per k-block): n1 if n2 > 0, else n1 / 2
  int n_tiles;         // weight tiles in all
  int cluster;         // CTAs per cluster: 1, or 2 (work units = tile pairs; activation boxes multicast, or mma2)
  int mma2;            // 1 (needs cluster == 2, w_fp16): tcgen05.mma.cta_group::2 over the pair, activation rows split
  int split;           // GemmSplit
  int splits;          // SPLIT_K: pieces per tile
  const GemmPiece* sched;  // device: [clusters][GEMM_MAX_PIECES] pieces, ended by pair = -1
  int n_cl;            // clusters of the launch (= rows of sched in use)
  int stages;
  int w_pre;           // weight tiles (pipeline stages) requested before griddepcontrol.wait
  int stg_bytes, stg_bufs;  // epilogue staging per warp: stg_bufs buffers of stg_bytes (2 x 4096, or 1 x 2048 to fit a stage more)
  int epi;             // GemmEpilogue
  int w_fp16;          // 1: the weight matrices already hold fp16 (af_convert_bf16_to_fp16); 0: bf16, converted per tile
  int out_f16;        // 0 = fp32 output (TMA stores through map_out), 2 = fp16 (16-byte global stores, fields below)
  void* out;           // fp16 output: element (feature f, middle m, token t) at out + t * out_ld_tok + m * out_ld_mid + f
  long long out_ld_tok, out_ld_mid;
  int out_features;    // features per middle index (multiple of 8): clips a ragged last tile
  void* partial;       // stream-K partials: fp32 [slot][512 tokens][128 features] written through map_part, or
  int part_f16;        // (part_f16, with fp16 outputs) raw fp16 staging images [slot][32-token chunk][lane quadrant][2 KB]
  int* flags;          // [grid] 0/1: set by the contributor, cleared by the owner (per stream: af_lib.cu StreamCtx)
};

#define AF_EPI_BAR_STR2(n) "bar.sync 1, " #n ";\n"
#define AF_EPI_BAR_STR(n) AF_EPI_BAR_STR2(n)
#define AF_EPI_BAR() asm volatile(AF_EPI_BAR_STR(AF_EPI_THREADS) ::: "memory")  /* the epilogue warps only */

#include "gemm_tcgen05_body.inl"

}  // namespace af
