// Persistent "layer chain" kernel for sm_100a: the projections of one decoder layer (Alg. 2) and the row
// stages between them run as PHASES of ONE launch, separated by in-kernel grid barriers instead of kernel boundaries:
//
//   [O proj -> slabs] | [x += slabs; RMSNorm] | [gate|up + SiLU*mul] | [down -> slabs] | [x += slabs; RMSNorm]
//                     | [QKV of the next layer -> slabs] | [slab reduce + RoPE + ring append  (FusedRoPEAndWriteKV)]
//                     | [attention of the next layer (attention_umma.cuh: tcgen05 units on the stage ring's shared memory)]
//
// One CTA per SM (74 two-CTA clusters), the warp roles of gemm_tcgen05.cuh (8 epilogue warps, one TMA producer, one MMA
// issuer), and one shared-memory stage ring that lives across the phases: the producer streams the WEIGHT tiles of the
// next projection into free stages while the current phase drains, synchronises and runs its row stage - weights never
// depend on activations (the packed step is one weight stream) - and only the ACTIVATION boxes of a stage wait
// for the grid barrier that publishes them.  Every projection stores plain fp16 pieces ("slabs", added up in fp32 by
// the row stage that follows, in slab order: deterministic) except gate|up, whose SiLU*mul epilogue needs complete sums
// and keeps the stream-K contributor -> owner fix-up (partials are exchanged in the epilogue threads' own register
// layout: the owner thread reads back exactly the 64 bytes its counterpart wrote, no shared-memory staging).
//
// Restrictions (the host falls back to the one-kernel-per-stage path otherwise): prepared fp16 weights with gate|up
// interleaved (AF_WEIGHTS_FP16_GU) or FP8 codes, T <= 1024 packed rows (above 512: two token chunks per piece, kTwo),
// d_model <= 4096, at least two weight tiles per projection.
#pragma once
#include "gemm_tcgen05.cuh"
#include "attention_umma.cuh"   // StepTables; the attention units of the chain's last phase

namespace af {

constexpr int CH_MAX_PHASES = 8;
constexpr int CH_MAX_MAPS = 12;
constexpr int CH_ROW_GROUPS = 2;          // row groups per CTA in a row stage (4 epilogue warps = 128 lanes each)
constexpr int CH_TRACE_SLOTS = 2 * CH_MAX_PHASES + 2;
constexpr int GEMM_MAX_SLABS_K = 4;       // slabs a row stage adds at most (= GEMM_MAX_SPLITS of af_lib.cu)
constexpr int QKV_MAX_SLABS_K = 4;        // slabs of the QKV projection (= QKV_MAX_SLABS of af_lib.cu; all are allocated)

enum ChainKind : int { CH_GEMM = 0, CH_ROWS = 1, CH_ROPE = 2, CH_ATTN = 3 };

struct ChainPhase {
  int kind;
  // ---- CH_GEMM ----
  int w_map[3], x_map;      // indices into ChainArgs::maps
  int part_rows, tiles_per_part, a_pair, n_tiles, num_kb;
  int epi;                  // EPI_STORE: every piece is stored as fp16 slab `mid`;  EPI_SWIGLU: stream-K with fix-up
  const GemmPiece* sched;   // [clusters][GEMM_MAX_PIECES]
  act_t* out;               // element (token t, slab s, part p, feature f) at out + s * out_ld_slab + t * out_ld_tok + p * part_rows + f
  long long out_ld_tok, out_ld_slab;
  int out_features;         // features per part (multiple of 8): clips a ragged last tile
  const float* scale[3];    // FP8 weights: per-output-channel fp32 scales of the parts (a_pair: [0] = gate, [1] = up)
  // ---- CH_ROWS: x[i,:] (= embeds[i,:] | += sum of slabs[s][i,:]);  xn[i,:] = fp16(RMSNorm(x[i,:]; gain)) unless gain == nullptr ----
  const void* src;          // nullptr: nothing to add; embed != 0: bf16 [T, D] embeddings; else fp16 slabs [n_slabs][.][D]
  int embed, n_slabs;
  long long slab_stride;    // elements between slabs
  const __nv_bfloat16* gain;
  act_t* xn;
  // ---- CH_ROPE: q|k|v = sum of the QKV slabs (src, slab_stride; slab counts per 256-feature tile pair in pair_slabs) ----
  const int* pair_slabs;
  act_t* q_out;             // [T, D] rotated queries
  act_t* kv_layer;          // ring, layer base: [2][R][H][C][hd]
};

struct ChainArgs {
  CUtensorMap maps[CH_MAX_MAPS];
  ChainPhase ph[CH_MAX_PHASES];
  int n_phases;
  int T, n1, n2;            // packed rows; UMMA N of the two token halves (n2 may be 0)
  int T0;                   // 0: one token chunk (T <= 512).  Else 512 < T <= 1024: every piece exists twice (GemmPiece::pad = token
                            // chunk 0 / 1, adjacent in its cluster's list, so the second pass re-reads its weight k-range from L2):
                            // chunk 0 = rows [0, T0), chunk 1 = rows [T0, T); n1, n2 describe one chunk
  int stages;
  int D;
  float eps;
  float* x;                 // residual stream fp32 [T, D] (hidden_out)
  unsigned long long* bar;  // grid barrier: arrival counter (see ld_acquire_gpu)
  int* flags;               // stream-K ready flags [grid]
  uint8_t* partial;         // stream-K partials (fp16, register layout) [slot][chunk][quadrant][2 KB]
  StepTables tb;            // row_pos / row_slot of the step (CH_ROPE)
  const float2* rope_tab;
  int H, hd, R, C;
  long long* trace;         // debug: [grid][CH_TRACE_SLOTS] globaltimer stamps, or nullptr
  int att_on;               // the LAST phase is CH_ATTN: attention of the layer whose q / k / v this launch has just produced
  AuArgs att;               // ... its arguments (attention_umma.cuh); the units' tiles reuse the stage ring
};

// FP8 weights (f4): a stage also holds the raw 8 KB E4M3 tile, which the epilogue warps widen to the fp16 UMMA tile
constexpr uint32_t CH_RAW_BYTES = GEMM_BM * GEMM_BK;
__device__ __forceinline__ uint32_t e4m3x2_to_f16x2(uint32_t two_codes) {   // exact: every E4M3 value is an fp16 value
  uint32_t r;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;\n" : "=r"(r) : "h"(static_cast<unsigned short>(two_codes)));
  return r;
}
__device__ __forceinline__ void mbar_arrive_leader_release(uint64_t* bar) {   // publishes this thread's (fenced) shared-memory writes to the pair's leader
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];\n" ::"r"(leader_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {   // acquire at cluster scope
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  }
}

// Grid barrier = one 64-bit arrival counter that only ever grows (it never wraps in practice and is a multiple of the
// grid size whenever no launch is in flight): barrier k of a launch is passed when count >= base + (k + 1) * grid.
__device__ __forceinline__ unsigned long long ld_acquire_gpu(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];\n" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_gpu_add(unsigned long long* p, unsigned long long v) {
  asm volatile("red.release.gpu.global.add.u64 [%0], %1;\n" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ int ld_acquire_cta_shared(const int* p) {
  int v;
  asm volatile("ld.acquire.cta.shared::cta.s32 %0, [%1];\n" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_cta_shared(int* p, int v) {
  asm volatile("st.release.cta.shared::cta.s32 [%0], %1;\n" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

// the 4 warps of a row group
#define AF_ROWGRP_BAR(g) asm volatile("bar.sync %0, 128;\n" ::"r"(2 + (g)) : "memory")

// Row stages of the chain, executed by the 8 epilogue warps of every CTA (two rows per CTA at a time, 4 warps = 128 lanes
// each).  Separate functions (their register allocation is independent of the GEMM epilogue's), arguments by value, and
// branch-free bodies: every 16-byte load of a lane's share of the row is in flight before the first use.
__device__ __forceinline__ void add_h8(const uint4& raw, bool on, float* o) {   // o[0..7] += the 8 fp16 values of raw (if on)
  const uint32_t w4[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w4[m]));
    o[2 * m] += on ? f.x : 0.f; o[2 * m + 1] += on ? f.y : 0.f;
  }
}

// x[i,:] (= embeds[i,:] | += sum of slabs[s][i,:]);  xn[i,:] = fp16(RMSNorm(x[i,:]; gain)) unless gain == nullptr
template <bool EMBED>
__device__ __noinline__ void chain_rows_phase(float* __restrict__ x, const void* __restrict__ src, int ns, long long slab_stride,
                                              const __nv_bfloat16* __restrict__ gain, act_t* __restrict__ xn, int D, float eps, int T,
                                              float (*row_red)[4], int cta, int n_cta, int warp, int lane) {
  const int grp = warp >> 2, gl = (warp & 3) * 32 + lane;    // lane 0..127 of the row group
  const int n_chunk = D >> 3;                                // 8-element chunks per row (<= 512: four per lane)
  const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);
  for (int i = cta * CH_ROW_GROUPS + grp; i < T; i += CH_ROW_GROUPS * n_cta) {   // (same trip count for the 4 warps of a group)
    float* xr = x + static_cast<size_t>(i) * D;
    const act_t* pr = reinterpret_cast<const act_t*>(src) + static_cast<size_t>(i) * D;
    float v[4][8];
    uint4 raw[4][GEMM_MAX_SLABS_K];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = gl + 128 * k;
      const bool ok = c < n_chunk;
      const int cc = ok ? c : 0;
      if (EMBED) {
        raw[k][0] = ok ? __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(src) + static_cast<size_t>(i) * D) + cc) : zero4;
      } else {
        const float4 lo = ok ? __ldcg(reinterpret_cast<const float4*>(xr) + 2 * cc) : make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 hi = ok ? __ldcg(reinterpret_cast<const float4*>(xr) + 2 * cc + 1) : make_float4(0.f, 0.f, 0.f, 0.f);
        v[k][0] = lo.x; v[k][1] = lo.y; v[k][2] = lo.z; v[k][3] = lo.w; v[k][4] = hi.x; v[k][5] = hi.y; v[k][6] = hi.z; v[k][7] = hi.w;
#pragma unroll
        for (int sl = 0; sl < GEMM_MAX_SLABS_K; ++sl)
          raw[k][sl] = (ok && sl < ns) ? __ldcg(reinterpret_cast<const uint4*>(pr + sl * slab_stride) + cc) : zero4;
      }
    }
    float ss = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = gl + 128 * k;
      const bool ok = c < n_chunk;
      if (EMBED) {
        const uint32_t w4[4] = {raw[k][0].x, raw[k][0].y, raw[k][0].z, raw[k][0].w};
#pragma unroll
        for (int m = 0; m < 4; ++m) { v[k][2 * m] = __uint_as_float(w4[m] << 16); v[k][2 * m + 1] = __uint_as_float(w4[m] & 0xffff0000u); }
      } else {
#pragma unroll
        for (int sl = 0; sl < GEMM_MAX_SLABS_K; ++sl) add_h8(raw[k][sl], true, v[k]);   // (absent slabs were loaded as zeros)
      }
      if (ok && (EMBED || ns > 0)) {
        __stcg(reinterpret_cast<float4*>(xr) + 2 * c, make_float4(v[k][0], v[k][1], v[k][2], v[k][3]));
        __stcg(reinterpret_cast<float4*>(xr) + 2 * c + 1, make_float4(v[k][4], v[k][5], v[k][6], v[k][7]));
      }
#pragma unroll
      for (int m = 0; m < 8; ++m) ss += v[k][m] * v[k][m];
    }
    if (gain) {
      uint4 graw[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) graw[k] = (gl + 128 * k < n_chunk) ? __ldg(reinterpret_cast<const uint4*>(gain) + gl + 128 * k) : zero4;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
      if (lane == 0) row_red[grp][warp & 3] = ss;
      AF_ROWGRP_BAR(grp);
      const float tot = row_red[grp][0] + row_red[grp][1] + row_red[grp][2] + row_red[grp][3];
      AF_ROWGRP_BAR(grp);
      const float inv = rsqrtf(tot / D + eps);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int c = gl + 128 * k;
        const uint32_t g4[4] = {graw[k].x, graw[k].y, graw[k].z, graw[k].w};
        uint4 o;
        uint32_t* op = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
        for (int m = 0; m < 4; ++m)
          op[m] = pack_act(v[k][2 * m] * inv * __uint_as_float(g4[m] << 16), v[k][2 * m + 1] * inv * __uint_as_float(g4[m] & 0xffff0000u));
        if (c < n_chunk) __stcg(reinterpret_cast<uint4*>(xn + static_cast<size_t>(i) * D) + c, o);
      }
    }
  }
}

// The fused slab-reduce + RoPE + ring-append stage (FusedRoPEAndWriteKV, Alg. 2 l.3): q|k|v of row i =
// sum of the QKV projection's slabs (slab counts per 256-feature tile pair in s_pair_slabs); q and k are rotated at the
// row's logical position in its own request (rotate-half pairing, table built in fp64); q goes to q_out, k and v straight
// to the row's ring slot.
template <bool kSplit>   // kSplit: fewer rows than row groups - a separate instantiation, the full-width step's code is untouched
__device__ __noinline__ void chain_rope_phase(const act_t* __restrict__ qkv, long long slab_stride, act_t* __restrict__ q_out,
                                              act_t* __restrict__ kv_layer, const int* __restrict__ row_pos,
                                              const int* __restrict__ row_slot, const float2* __restrict__ rope_tab, int H, int hd,
                                              int R, int C, int D, int T, const int* s_pair_slabs, int cta, int n_cta, int warp, int lane) {
  const int grp = warp >> 2, gl = (warp & 3) * 32 + lane;
  const int half = hd >> 1, per_head = half / 8;
  const int n_qk = 2 * H * per_head, n_v = D / 8;
  // A row's items are walked 256 at a time (two per lane, every load in flight before the first use): D / 2048 passes for
  // q | k plus as many for v, each an L2 round trip.  With fewer rows than row groups (decode-only steps, short prefills) a
  // row is split over up to 4 groups, each taking every n_parts-th pass.
  const int n_grp = CH_ROW_GROUPS * n_cta;
  const int n_parts = kSplit ? min(4, n_grp / T) : 1;
  const int qk_passes = (n_qk + 255) / 256;
  for (int unit = cta * CH_ROW_GROUPS + grp; unit < T * n_parts; unit += n_grp) {
    const int i = unit / n_parts, part = unit - i * n_parts;
    const int pos = __ldg(row_pos + i), gslot = __ldg(row_slot + i);
    const int req = gslot / C, slot = gslot - req * C;
    const act_t* src = qkv + static_cast<size_t>(i) * 3 * D;
    const float2* tab = rope_tab + static_cast<size_t>(pos) * half;
    const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);
    for (int w0 = gl + 256 * part; w0 < n_qk; w0 += 256 * n_parts) {   // q, k: two (head, 8-element) items per lane at a time
      uint4 rlo[2][QKV_MAX_SLABS_K], rhi[2][QKV_MAX_SLABS_K];
      float4 cs[2][4];
      int colv[2], hv[2], cv[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int w = w0 + 128 * u < n_qk ? w0 + 128 * u : w0;
        const int which = w / (H * per_head);           // 0 = q, 1 = k
        const int rem = w - which * H * per_head;
        hv[u] = rem / per_head; cv[u] = (rem - hv[u] * per_head) * 8;
        colv[u] = which * D + hv[u] * hd + cv[u];
        const int ns = s_pair_slabs[colv[u] / (2 * GEMM_BM)];   // (col and col + half lie in the same 128-feature tile)
#pragma unroll
        for (int sl = 0; sl < QKV_MAX_SLABS_K; ++sl) {
          rlo[u][sl] = sl < ns ? __ldcg(reinterpret_cast<const uint4*>(src + sl * slab_stride + colv[u])) : zero4;
          rhi[u][sl] = sl < ns ? __ldcg(reinterpret_cast<const uint4*>(src + sl * slab_stride + colv[u] + half)) : zero4;
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) cs[u][e] = __ldg(reinterpret_cast<const float4*>(tab + cv[u]) + e);   // (cos, sin) of 2 elements each
      }
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        float lo[8], hi[8];
#pragma unroll
        for (int m = 0; m < 8; ++m) { lo[m] = 0.f; hi[m] = 0.f; }
#pragma unroll
        for (int sl = 0; sl < QKV_MAX_SLABS_K; ++sl) { add_h8(rlo[u][sl], true, lo); add_h8(rhi[u][sl], true, hi); }
        uint4 out_lo, out_hi;
        uint32_t* ol = reinterpret_cast<uint32_t*>(&out_lo);
        uint32_t* oh = reinterpret_cast<uint32_t*>(&out_hi);
#pragma unroll
        for (int e = 0; e < 8; e += 2) {
          const float4 t4 = cs[u][e >> 1];                // cos(e), sin(e), cos(e + 1), sin(e + 1)
          ol[e >> 1] = pack_act(lo[e] * t4.x - hi[e] * t4.y, lo[e + 1] * t4.z - hi[e + 1] * t4.w);
          oh[e >> 1] = pack_act(hi[e] * t4.x + lo[e] * t4.y, hi[e + 1] * t4.z + lo[e + 1] * t4.w);
        }
        const bool is_q = colv[u] < D;
        act_t* dst = is_q ? q_out + static_cast<size_t>(i) * D + hv[u] * hd + cv[u]
                          : kv_layer + ((static_cast<size_t>(0 * R + req) * H + hv[u]) * C + slot) * hd + cv[u];
        if (w0 + 128 * u < n_qk) {
          *reinterpret_cast<uint4*>(dst) = out_lo;
          *reinterpret_cast<uint4*>(dst + half) = out_hi;
        }
      }
    }
    const int v_first = ((part - qk_passes) % n_parts + n_parts) % n_parts;   // v's pass k is pass qk_passes + k of the row
    for (int w0 = gl + 256 * v_first; w0 < n_v; w0 += 256 * n_parts) {   // v: two 8-element items per lane at a time
      uint4 rv[2][QKV_MAX_SLABS_K];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int w = w0 + 128 * u < n_v ? w0 + 128 * u : w0;
        const int ns = s_pair_slabs[(2 * D + w * 8) / (2 * GEMM_BM)];
#pragma unroll
        for (int sl = 0; sl < QKV_MAX_SLABS_K; ++sl)
          rv[u][sl] = sl < ns ? __ldcg(reinterpret_cast<const uint4*>(src + sl * slab_stride + 2 * D + w * 8)) : zero4;
      }
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int w = w0 + 128 * u;
        float o[8];
#pragma unroll
        for (int m = 0; m < 8; ++m) o[m] = 0.f;
#pragma unroll
        for (int sl = 0; sl < QKV_MAX_SLABS_K; ++sl) add_h8(rv[u][sl], true, o);
        const int h = (w * 8) / hd, c = (w * 8) - h * hd;
        uint4 v;
        v.x = pack_act(o[0], o[1]); v.y = pack_act(o[2], o[3]); v.z = pack_act(o[4], o[5]); v.w = pack_act(o[6], o[7]);
        if (w < n_v) *reinterpret_cast<uint4*>(kv_layer + ((static_cast<size_t>(1 * R + req) * H + h) * C + slot) * hd + c) = v;
      }
    }
  }
}

// CH_ATTN on the 8 epilogue warps (a function of its own: its register allocation is independent of the GEMM epilogue's)
// (the shared-memory pointers are rebuilt from the dynamic allocation here, not passed in: through a call boundary they would
// be generic pointers and every P store / table read a generic access; the arguments travel by value)
__device__ __noinline__ void chain_attn_phase(uint32_t tmem, const AuArgs a, const AuLists* lists, int cta, int n_cta, int tid) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  AuAux* x = reinterpret_cast<AuAux*>(tiles + AU_TILE_BYTES);
  long long* trace = a.trace;
  AU_STAMP(0);
  au_workers(*x, *lists, tiles, tmem, a, cta, n_cta, tid);
}

// kTwo: 512 < T <= 1024, two token chunks per piece (ChainArgs::T0); a separate instantiation so that the one-chunk kernel
// - the benchmark path - carries none of the chunk arithmetic (measured: 4 % of the step when it was a runtime branch).
template <bool kFp8, bool kTwo>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
layer_chain_kernel(const __grid_constant__ ChainArgs a) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int T0 = kTwo ? a.T0 : 0;
  const int n_pad = a.n1 + a.n2;
  constexpr uint32_t a_bytes = GEMM_BM * GEMM_BK * 2;
  const uint32_t b_bytes = static_cast<uint32_t>(n_pad / 2) * GEMM_BK * 2;   // this CTA's half of the activation rows
  const uint32_t stage_bytes = a_bytes + b_bytes;   // [fp16 weight tile (FP8: the raw 8 KB tile lands in its upper half)][activation boxes]
  uint8_t* xch = tiles + static_cast<size_t>(a.stages) * stage_bytes;         // 8 x 2 KB epilogue staging
  AuAux* ax = reinterpret_cast<AuAux*>(tiles + AU_TILE_BYTES);                // CH_ATTN: the units' small state, behind their tiles

  // full_bar: the stage's TMA loads have landed (FP8: the activation boxes only; the raw weight tile lands on this CTA's
  // own wfull_bar and conv_bar, on the pair's leader, counts the epilogue warps of BOTH CTAs that have widened their tile)
  __shared__ uint64_t full_bar[GEMM_MAX_STAGES], empty_bar[GEMM_MAX_STAGES], tmem_full_bar, tmem_empty_bar;
  __shared__ uint64_t wfull_bar[GEMM_MAX_STAGES], conv_bar[GEMM_MAX_STAGES];
  __shared__ uint32_t tmem_base_smem;
  __shared__ int deps_done;                         // grid barriers this CTA has passed (published to the producer)
  __shared__ float row_red[CH_ROW_GROUPS][4];
  __shared__ int s_pair_slabs[64];
  __shared__ AuLists att_lists;                     // CH_ATTN: the step's unit lists, built at kernel start

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cta = blockIdx.x, n_cta = gridDim.x;
  const int crank = static_cast<int>(cluster_ctarank());
  const int cl = cta >> 1;
  long long* trace = a.trace ? a.trace + static_cast<size_t>(cta) * CH_TRACE_SLOTS : nullptr;

  if (warp == GEMM_EPI_WARPS && lane == 0) {
    for (int s = 0; s < a.stages; ++s) {
      mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1);
      mbar_init(&wfull_bar[s], 1); mbar_init(&conv_bar[s], GEMM_EPI_WARPS);   // 4 warps of each CTA of the pair
    }
    mbar_init(&tmem_full_bar, 1);
    mbar_init(&tmem_empty_bar, 2 * GEMM_EPI_WARPS);   // the leader waits for both CTAs' drains
    fence_barrier_init();
    deps_done = 0;
  }
  if (warp == GEMM_EPI_WARPS + 1) tmem_alloc_cg2(&tmem_base_smem, GEMM_TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  cluster_sync();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  pdl_launch_dependents();

  auto get_piece = [&](const GemmPiece* list, int i) {
    GemmPiece pc;
    const int4* src = reinterpret_cast<const int4*>(list + i);
    *reinterpret_cast<int4*>(&pc) = __ldg(src);
    *(reinterpret_cast<int4*>(&pc) + 1) = __ldg(src + 1);
    return pc;
  };

  if (warp == GEMM_EPI_WARPS) {
    // ================================ TMA producer ================================
    // Two cursors over the same sequence of (phase, piece, k-block) units: the WEIGHT cursor runs ahead as far as the
    // stage ring allows; the ACTIVATION cursor follows and stops at a phase until that phase's input has been
    // published (deps_done, raised by this CTA's epilogue after the grid barrier; phase 0: griddepcontrol.wait).
    if (lane == 0) {
      const uint64_t pol_w = T0 > 0 ? policy_evict_last() : policy_evict_first();   // (two token chunks: the second pass re-reads the k-range from L2)
      const uint64_t pol_x = policy_evict_last();
      // A cursor walks the (phase, piece, k-block) units of this cluster in order; all of its state is in registers.
      struct Cursor { int ph, pi, kb, kb1, row, tok0; const CUtensorMap* wmap; const CUtensorMap* xmap; const GemmPiece* list; bool more; };
      auto next_piece = [&](Cursor& c) {   // move to the next (phase, piece) that has k-blocks
        while (true) {
          if (c.ph >= 0 && c.pi + 1 < GEMM_MAX_PIECES) {
            const GemmPiece pc = get_piece(c.list, ++c.pi);
            if (pc.pair >= 0) {
              if (pc.kb1 <= pc.kb0) continue;
              const ChainPhase& P = a.ph[c.ph];
              const int tile = min(pc.pair * 2 + crank, P.n_tiles - 1);   // (an odd tile count: reload the last)
              int part = 0;
              if (!P.a_pair) part = tile / P.tiles_per_part;
              c.wmap = &a.maps[P.w_map[part]];
              c.row = P.a_pair ? tile * GEMM_BM : (tile - part * P.tiles_per_part) * GEMM_BM;
              c.kb = pc.kb0; c.kb1 = pc.kb1;
              c.tok0 = kTwo ? pc.pad * T0 : 0;
              return;
            }
          }
          do { ++c.ph; } while (c.ph < a.n_phases && a.ph[c.ph].kind != CH_GEMM);
          if (c.ph >= a.n_phases) { c.more = false; return; }
          c.list = a.ph[c.ph].sched + static_cast<size_t>(cl) * GEMM_MAX_PIECES;
          c.xmap = &a.maps[a.ph[c.ph].x_map];
          c.pi = -1;
        }
      };
      auto advance = [&](Cursor& c) { if (++c.kb == c.kb1) next_piece(c); };
      const int h1 = a.n1 / 2;
      auto load_w = [&](const Cursor& c, int stage) {
        if (kFp8) {   // raw E4M3 tile -> this CTA's own barrier (its epilogue warps widen it); activations -> the leader's
          if (crank == 0) mbar_arrive_expect_tx(&full_bar[stage], 2 * b_bytes);
          mbar_arrive_expect_tx(&wfull_bar[stage], CH_RAW_BYTES);
          tma_load_2d(tiles + static_cast<size_t>(stage) * stage_bytes + CH_RAW_BYTES, c.wmap, &wfull_bar[stage], c.kb * GEMM_BK, c.row, pol_w);
        } else {
          if (crank == 0) mbar_arrive_expect_tx(&full_bar[stage], 2 * stage_bytes);
          tma_load_2d_cg2(tiles + static_cast<size_t>(stage) * stage_bytes, c.wmap, &full_bar[stage], c.kb * GEMM_BK, c.row, pol_w);
        }
      };
      auto load_x = [&](const Cursor& c, int stage) {
        uint8_t* sb = tiles + static_cast<size_t>(stage) * stage_bytes + a_bytes;
        tma_load_2d_cg2(sb, c.xmap, &full_bar[stage], c.kb * GEMM_BK, c.tok0 + crank * h1, pol_x);
        if (a.n2 > 0)
          tma_load_2d_cg2(sb + static_cast<size_t>(h1) * GEMM_BK * 2, c.xmap, &full_bar[stage], c.kb * GEMM_BK, c.tok0 + a.n1 + crank * h1, pol_x);
      };
      Cursor w{-1, GEMM_MAX_PIECES, 0, 0, 0, 0, nullptr, nullptr, nullptr, true};
      next_piece(w);
      Cursor x = w;                      // the activation cursor: equal to w in lock step, behind it at a phase boundary
      int st_w = 0, st_x = 0, lag = 0;   // lag = stages that hold weights but not yet their activations
      uint32_t par_w = 0;
      int deps_seen = 0;
      bool pdl_done = false;
      while (w.more || lag > 0) {
        if (lag == 0 && deps_seen >= w.ph && pdl_done) {
          // ---- lock step (the steady state of a phase): one stage = weight tile + activation boxes ----
          mbar_wait(&empty_bar[st_w], par_w ^ 1);
          load_w(w, st_w);
          load_x(w, st_w);
          advance(w);
          if (++st_w == a.stages) { st_w = 0; par_w ^= 1; }
          continue;
        }
        if (lag == 0) { x = w; st_x = st_w; }
        // ---- phase boundary: weights run ahead into free stages, activations follow once their phase is published ----
        bool w_issued = false;
        if (w.more && lag < a.stages && mbar_try_wait(&empty_bar[st_w], par_w ^ 1)) {
          load_w(w, st_w);
          advance(w);
          if (++st_w == a.stages) { st_w = 0; par_w ^= 1; }
          ++lag;
          w_issued = true;
        }
        if (lag > 0) {
          if (deps_seen < x.ph) {
            deps_seen = ld_acquire_cta_shared(&deps_done);
            if (deps_seen >= x.ph) fence_proxy_async_all();   // the published rows were written through the generic proxy
          }
          if (deps_seen >= x.ph) {
            if (!pdl_done) {
              if (w_issued) continue;                          // keep prefetching weights before blocking on the previous grid
              pdl_wait();
              pdl_done = true;
            }
            load_x(x, st_x);
            advance(x);
            if (++st_x == a.stages) st_x = 0;
            --lag;
          }
        }
      }
      if (!pdl_done) pdl_wait();
    }
  } else if (warp == GEMM_EPI_WARPS + 1) {
    // ================================ MMA issuer (one thread of the pair's leader) ================================
    if (lane == 0 && crank == 0) {
      const uint32_t idesc1 = umma_idesc_f16(2 * GEMM_BM, a.n1);
      const uint32_t idesc2 = umma_idesc_f16(2 * GEMM_BM, a.n2 > 0 ? a.n2 : 16);
      int stage = 0;
      uint32_t phase = 0, acc_phase = 0;
      for (int ph = 0; ph < a.n_phases; ++ph) {
        if (a.ph[ph].kind != CH_GEMM) continue;
        const GemmPiece* list = a.ph[ph].sched + static_cast<size_t>(cl) * GEMM_MAX_PIECES;
        for (int pi = 0; pi < GEMM_MAX_PIECES; ++pi) {
          const GemmPiece pc = get_piece(list, pi);
          if (pc.pair < 0) break;
          if (pc.kb1 <= pc.kb0) continue;
          mbar_wait(&tmem_empty_bar, acc_phase ^ 1);
          tc_fence_after();
          for (int kb = pc.kb0; kb < pc.kb1; ++kb) {
            mbar_wait(&full_bar[stage], phase);
            if (kFp8) mbar_wait(&conv_bar[stage], phase);   // both CTAs' weight tiles have been widened to fp16
            tc_fence_after();
            const uint32_t sa = smem_u32(tiles + static_cast<size_t>(stage) * stage_bytes);
            const uint32_t sb = sa + a_bytes;
            const uint64_t da = umma_smem_desc_sw128(sa);
            const uint64_t db1 = umma_smem_desc_sw128(sb);
            const uint64_t db2 = umma_smem_desc_sw128(sb + (a.n1 / 2) * GEMM_BK * 2);
#pragma unroll
            for (int k = 0; k < GEMM_BK / 16; ++k) {
              const uint32_t accum = (kb > pc.kb0 || k > 0) ? 1u : 0u;
              umma_f16_cg2(tmem_base, da + 2 * k, db1 + 2 * k, idesc1, accum);
              if (a.n2 > 0) umma_f16_cg2(tmem_base + a.n1, da + 2 * k, db2 + 2 * k, idesc2, accum);
            }
            umma_commit_cg2_mc(&empty_bar[stage], 0x3);
            if (++stage == a.stages) { stage = 0; phase ^= 1; }
          }
          umma_commit_cg2_mc(&tmem_full_bar, 0x3);
          acc_phase ^= 1;
        }
      }
    }
    // CH_ATTN (always the last phase): every CTA issues its own units' MMAs (cta_group::1) - nothing below waits on it
    // (its barriers live in the epilogue staging area: they are initialised at the grid barrier before the phase, see below)
    if (lane == 0 && a.att_on) {
      while (ld_acquire_cta_shared(&deps_done) < a.n_phases - 1) {}
      au_mma_loop(*ax, tiles, tmem_base);
    }
  } else {
    // ================================ epilogue warps 0..7: drains, row stages, grid barriers ================================
    const int quad = warp & 3, par = warp >> 2;
    const int etid = threadIdx.x;   // 0..255
    uint8_t* stg_base = xch + warp * 2048;
    const uint32_t frag_off64 = (lane & 7) * 64 + (((lane >> 3) ^ ((lane & 7) >> 1)) << 4);
    const uint32_t frag_off32 = ((lane >> 4) * 8 + (lane & 7)) * 32 + ((((lane >> 3) & 1) ^ ((lane & 7) >> 2)) << 4);
    const uint32_t rb_off64 = (lane >> 2) * 64 + (((lane & 3) ^ ((lane >> 3) & 3)) << 4);
    const uint32_t rb_off32 = (lane >> 1) * 32 + (((lane & 1) ^ ((lane >> 3) & 1)) << 4);
    pdl_wait();
    unsigned long long bar_target = 0;
    if (etid == 0) {
      // arrivals of faster CTAs at this launch's first barrier may already be counted: round down to the launch's base
      bar_target = ld_acquire_gpu(a.bar) / static_cast<unsigned>(n_cta) * static_cast<unsigned>(n_cta);
      if (trace) trace[0] = static_cast<long long>(globaltimer_ns());
    }
    for (int ph = 0; ph < a.n_phases; ++ph)   // slab counts of the RoPE stage's tile pairs: one shared-memory lookup per item
      if (a.ph[ph].kind == CH_ROPE)
        for (int i = etid; i < 3 * a.D / (2 * GEMM_BM) && i < 64; i += GEMM_EPI_WARPS * 32) s_pair_slabs[i] = __ldg(a.ph[ph].pair_slabs + i);
    AF_EPI_BAR();
    if (a.att_on) au_build_lists(att_lists, a.att.tb, a.att.n_segs, etid);   // (the warps would wait for the first accumulator anyway)
    uint32_t acc_phase = 0, cphase = 0;
    int n_bar = 0, cstage = 0, cunit = 0;

    for (int ph = 0; ph < a.n_phases; ++ph) {
      const ChainPhase& P = a.ph[ph];
      if (P.kind == CH_GEMM) {
        const GemmPiece* list = P.sched + static_cast<size_t>(cl) * GEMM_MAX_PIECES;
        for (int pi = 0; pi < GEMM_MAX_PIECES; ++pi) {
          const GemmPiece pc = get_piece(list, pi);
          if (pc.pair < 0) break;
          const bool has_mma = pc.kb1 > pc.kb0;
          const int tile = pc.pair * 2 + crank;
          const bool tile_valid = tile < P.n_tiles;
          if (kFp8) {
            // ---- widen this piece's raw E4M3 weight tiles to the fp16 UMMA tile (K-major, 128-byte swizzle), stage by stage
            //      as they land.  The two groups of 4 warps take alternate stages (two conversions in flight). ----
            const int cg = warp >> 2, ct = (warp & 3) * 32 + lane;   // thread 0..127 of its group
            for (int kb = pc.kb0; kb < pc.kb1; ++kb) {
              if ((cunit & 1) == cg) {
                mbar_wait(&wfull_bar[cstage], cphase);
                uint8_t* sbase = tiles + static_cast<size_t>(cstage) * stage_bytes;
                const uint4* raw = reinterpret_cast<const uint4*>(sbase + CH_RAW_BYTES);   // upper half of the 16 KB fp16 tile
                // 16-byte chunk id = i * 128 + ct (a warp reads 512 contiguous bytes: no bank conflicts) = 16 codes of row
                // id / 4, which become fp16 chunks 2 (id % 4) and 2 (id % 4) + 1 of that row in the swizzled tile
                uint4 c4[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) c4[i] = raw[i * 128 + ct];
                AF_ROWGRP_BAR(cg);   // in-place expansion: every raw chunk is in registers before the first fp16 chunk is written
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  const int id = i * 128 + ct, r = id >> 2, cc = (id & 3) * 2;
                  uint4 o0, o1;
                  o0.x = e4m3x2_to_f16x2(c4[i].x); o0.y = e4m3x2_to_f16x2(c4[i].x >> 16);
                  o0.z = e4m3x2_to_f16x2(c4[i].y); o0.w = e4m3x2_to_f16x2(c4[i].y >> 16);
                  o1.x = e4m3x2_to_f16x2(c4[i].z); o1.y = e4m3x2_to_f16x2(c4[i].z >> 16);
                  o1.z = e4m3x2_to_f16x2(c4[i].w); o1.w = e4m3x2_to_f16x2(c4[i].w >> 16);
                  *reinterpret_cast<uint4*>(sbase + r * 128 + ((cc ^ (r & 7)) << 4)) = o0;
                  *reinterpret_cast<uint4*>(sbase + r * 128 + (((cc + 1) ^ (r & 7)) << 4)) = o1;
                }
                // Generic-proxy writes -> the tensor core's (async-proxy) reads, possibly issued from the peer CTA: the proxy
                // fence completes this thread's shared-memory writes towards the async proxy before the arrive is issued; the
                // arrive itself is relaxed (a cluster-scope release costs ~1000 cycles per stage here - measured: 2x the
                // whole step), the leader's wait acquires at cluster scope.
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive_leader(&conv_bar[cstage]);
              }
              ++cunit;
              if (++cstage == a.stages) { cstage = 0; cphase ^= 1; }
            }
          }
          const bool contributor = pc.kind == PK_CONTRIB;
          const int chunk = kTwo ? pc.pad : 0, tok0 = chunk * T0;                      // token chunk of this piece (0 unless T > 512)
          const int Tv = T0 > 0 ? (chunk ? a.T - T0 : T0) : a.T;        // its valid rows
          const int nch = T0 > 0 ? 2 : 1;
          const int my_slot = (pc.slot * nch + chunk) * 2 + crank;           // partial / flag slot: per (cluster, chunk, CTA of the pair)
          int n_contrib = 0, c_first = 0;
          if (pc.kind == PK_OWNER) {
            c_first = pc.slot; n_contrib = pc.n_contrib;
            if (etid < n_contrib) {
              volatile int* f = a.flags + ((c_first + etid) * nch + chunk) * 2 + crank;
              SpinGuard sg;
              while (*f == 0) sg.poll();
              *f = 0;   // one consumer per flag: ready for the next use (graph-replay safe)
              __threadfence();
            }
            AF_EPI_BAR();
          }
          int f0, part = 0;
          if (P.a_pair) f0 = tile * 64 + quad * 16;
          else { part = tile / P.tiles_per_part; f0 = (tile - part * P.tiles_per_part) * GEMM_BM + quad * 32; }
          const int st_sh = P.epi == EPI_SWIGLU ? 1 : 2;
          const int st_feat = f0 + 8 * (lane & ((1 << st_sh) - 1)), st_tok = lane >> st_sh;
          const bool st_ok = tile_valid && st_feat < P.out_features;
          act_t* const st_ptr = P.out + static_cast<size_t>(P.epi == EPI_SWIGLU ? 0 : pc.mid) * P.out_ld_slab +
                                static_cast<size_t>(part) * P.part_rows + st_feat + static_cast<size_t>(tok0 + st_tok) * P.out_ld_tok;
          // partial exchange (stream-K): thread-private 64 bytes per 32-token chunk, in the epilogue's register layout
          auto part_ptr = [&](int slot, int c0) {
            return a.partial + (static_cast<size_t>(slot) * (GEMM_MAX_TOK / 32) * 4 + (c0 >> 5) * 4 + quad) * 2048 + lane * 16;
          };
          // FP8: per-output-channel scales of this thread's four accumulator rows (TMEM lanes lane/4, +8, +16, +24 of the quadrant)
          float sc4[4] = {1.f, 1.f, 1.f, 1.f};
          if (kFp8) {
            if (P.a_pair) {   // lanes [0,16) = gate rows, [16,32) = up rows of features tile * 64 + quad * 16 + ..
              const int f = tile * 64 + quad * 16 + (lane >> 2);
              sc4[0] = f < P.out_features ? __ldg(P.scale[0] + f) : 0.f;     sc4[1] = f + 8 < P.out_features ? __ldg(P.scale[0] + f + 8) : 0.f;
              sc4[2] = f < P.out_features ? __ldg(P.scale[1] + f) : 0.f;     sc4[3] = f + 8 < P.out_features ? __ldg(P.scale[1] + f + 8) : 0.f;
            } else {
              const int fl = f0 + (lane >> 2);
#pragma unroll
              for (int j = 0; j < 4; ++j) sc4[j] = (tile_valid && fl + 8 * j < P.out_features) ? __ldg(P.scale[part] + fl + 8 * j) : 0.f;
            }
          }
          auto apply_scale = [&](float* w) {
            if (kFp8) {
#pragma unroll
              for (int g = 0; g < 4; ++g) {
                w[4 * g] *= sc4[0]; w[4 * g + 1] *= sc4[0]; w[4 * g + 2] *= sc4[1]; w[4 * g + 3] *= sc4[1];
                w[16 + 4 * g] *= sc4[2]; w[16 + 4 * g + 1] *= sc4[2]; w[16 + 4 * g + 2] *= sc4[3]; w[16 + 4 * g + 3] *= sc4[3];
              }
            }
          };
          if (has_mma) mbar_wait(&tmem_full_bar, acc_phase);
          tc_fence_after();

          auto issue = [&](int c0, float* w) {
            if (has_mma) {
              const uint32_t ta = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + c0;
              tmem_ld_frag32f(ta, w);
              tmem_ld_frag32f(ta + (16u << 16), w + 16);
            } else {
#pragma unroll
              for (int j = 0; j < 32; ++j) w[j] = 0.f;
            }
          };
          auto fix_load = [&](int c, int c0, uint4* q) {   // contributor c's partial of this thread's chunk
            const uint8_t* src = part_ptr(((c_first + c) * nch + chunk) * 2 + crank, c0);
#pragma unroll
            for (int g = 0; g < 4; ++g) q[g] = __ldcg(reinterpret_cast<const uint4*>(src + g * 512));
          };
          auto fix_add = [&](const uint4* q, float* v) {
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              const uint32_t w4[4] = {q[g].x, q[g].y, q[g].z, q[g].w};
#pragma unroll
              for (int m = 0; m < 4; ++m) {
                const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w4[m]));
                v[8 * g + 2 * m] += f.x; v[8 * g + 2 * m + 1] += f.y;
              }
            }
          };
          auto finish_chunk = [&](int c0, float* v) {
            if (contributor) {
              uint8_t* dst = part_ptr(my_slot, c0);
#pragma unroll
              for (int g = 0; g < 4; ++g) {
                uint4 q;
                q.x = pack_act(v[8 * g], v[8 * g + 1]); q.y = pack_act(v[8 * g + 2], v[8 * g + 3]);
                q.z = pack_act(v[8 * g + 4], v[8 * g + 5]); q.w = pack_act(v[8 * g + 6], v[8 * g + 7]);
                if (tile_valid) __stcg(reinterpret_cast<uint4*>(dst + g * 512), q);
              }
            } else if (P.epi == EPI_STORE) {
              __syncwarp();
              const uint32_t sa = smem_u32(stg_base);
#pragma unroll
              for (int g = 0; g < 4; ++g)
                stmatrix_x4_trans(sa + frag_off64 + g * 512, pack_act(v[4 * g], v[4 * g + 1]), pack_act(v[4 * g + 2], v[4 * g + 3]),
                                  pack_act(v[16 + 4 * g], v[16 + 4 * g + 1]), pack_act(v[16 + 4 * g + 2], v[16 + 4 * g + 3]));
              __syncwarp();
              act_t* dst = st_ptr + static_cast<size_t>(c0) * P.out_ld_tok;
              const int n_ok = Tv - c0 - st_tok;
#pragma unroll
              for (int g = 0; g < 4; ++g)
                if (st_ok && 8 * g < n_ok)
                  __stcg(reinterpret_cast<uint4*>(dst + static_cast<size_t>(8 * g) * P.out_ld_tok), lds128(sa + rb_off64 + g * 512));
            } else {   // EPI_SWIGLU: v[j] = gate, v[16 + j] = up of one (feature, token)
              uint32_t h[8];
#pragma unroll
              for (int j = 0; j < 16; j += 2) {
                const float g0 = v[j], g1 = v[j + 1];
                const float h0 = __fdividef(g0, 1.f + __expf(-g0)) * v[16 + j], h1 = __fdividef(g1, 1.f + __expf(-g1)) * v[17 + j];
                h[j >> 1] = pack_act(h0, h1);
              }
              __syncwarp();
              const uint32_t sa = smem_u32(stg_base);
              stmatrix_x4_trans(sa + frag_off32, h[0], h[1], h[2], h[3]);
              stmatrix_x4_trans(sa + frag_off32 + 512, h[4], h[5], h[6], h[7]);
              __syncwarp();
              act_t* dst = st_ptr + static_cast<size_t>(c0) * P.out_ld_tok;
              const int n_ok = Tv - c0 - st_tok;
#pragma unroll
              for (int j = 0; j < 2; ++j)
                if (st_ok && 16 * j < n_ok)
                  __stcg(reinterpret_cast<uint4*>(dst + static_cast<size_t>(16 * j) * P.out_ld_tok), lds128(sa + rb_off32 + j * 512));
            }
          };
          // software pipeline over this warp's 32-token chunks: the TMEM load (and the first contributor's partial) of
          // chunk i + 1 is in flight while chunk i is converted and stored
          {
            float v[32], vb[32];
            uint4 q[4];
            auto in_range = [&](int c0) { return c0 < n_pad && c0 < Tv; };
            auto step = [&](int c0, float* cur, float* nxt) {
              tmem_ld_wait();
              apply_scale(cur);     // (before the fix-up adds and every store: partials and slabs carry scaled sums)
              if (n_contrib > 0) {
                fix_add(q, cur);
                for (int c = 1; c < n_contrib; ++c) { uint4 q2[4]; fix_load(c, c0, q2); fix_add(q2, cur); }
              }
              const int cn = c0 + GEMM_BLK;
              if (in_range(cn)) { issue(cn, nxt); if (n_contrib > 0) fix_load(0, cn, q); }
              finish_chunk(c0, cur);
            };
            int c0 = 32 * par;
            if (in_range(c0)) { issue(c0, v); if (n_contrib > 0) fix_load(0, c0, q); }
            while (in_range(c0)) {
              step(c0, v, vb);
              c0 += GEMM_BLK;
              if (!in_range(c0)) break;
              step(c0, vb, v);
              c0 += GEMM_BLK;
            }
          }
          tc_fence_before();
          __syncwarp();
          if (lane == 0 && has_mma) mbar_arrive_leader(&tmem_empty_bar);
          if (contributor) {
            __threadfence();
            AF_EPI_BAR();
            if (etid == 0) {
              __threadfence();
              atomicExch(a.flags + my_slot, 1);
            }
          }
          if (has_mma) acc_phase ^= 1;
        }
      } else if (P.kind == CH_ROWS) {
        const int ns = (P.src && !P.embed) ? P.n_slabs : 0;
        if (P.embed) chain_rows_phase<true>(a.x, P.src, 0, 0, P.gain, P.xn, a.D, a.eps, a.T, row_red, cta, n_cta, warp, lane);
        else chain_rows_phase<false>(a.x, P.src ? P.src : a.x, ns, P.slab_stride, P.gain, P.xn, a.D, a.eps, a.T, row_red, cta, n_cta, warp, lane);
      } else if (P.kind == CH_ROPE) {
        if (2 * a.T <= CH_ROW_GROUPS * n_cta)
          chain_rope_phase<true>(reinterpret_cast<const act_t*>(P.src), P.slab_stride, P.q_out, P.kv_layer, a.tb.row_pos, a.tb.row_slot,
                                 a.rope_tab, a.H, a.hd, a.R, a.C, a.D, a.T, s_pair_slabs, cta, n_cta, warp, lane);
        else
          chain_rope_phase<false>(reinterpret_cast<const act_t*>(P.src), P.slab_stride, P.q_out, P.kv_layer, a.tb.row_pos, a.tb.row_slot,
                                  a.rope_tab, a.H, a.hd, a.R, a.C, a.D, a.T, s_pair_slabs, cta, n_cta, warp, lane);
      } else {
        chain_attn_phase(tmem_base, a.att, &att_lists, cta, n_cta, etid);
      }
      if (etid == 0 && trace) trace[1 + 2 * ph] = static_cast<long long>(globaltimer_ns());
      // ---- grid barrier: everything this phase wrote is visible to every CTA before the next phase reads it ----
      if (ph + 1 < a.n_phases) {
        AF_EPI_BAR();
        if (etid == 0) {
          bar_target += static_cast<unsigned>(n_cta);
          red_release_gpu_add(a.bar, 1ull);       // (release: cumulative over what the CTA's threads wrote before bar.sync)
          SpinGuard sg;
          while (ld_acquire_gpu(a.bar) < bar_target) sg.poll();
          fence_proxy_async_all();
          if (a.att_on && ph + 2 == a.n_phases) {   // the next phase is CH_ATTN: its mbarriers (the staging area is free from here on)
            au_init_barriers(*ax);
            fence_barrier_init();
          }
          st_release_cta_shared(&deps_done, ++n_bar);
          if (trace) trace[2 + 2 * ph] = static_cast<long long>(globaltimer_ns());
        }
        AF_EPI_BAR();
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync();
  if (warp == GEMM_EPI_WARPS + 1) {
    tc_fence_after();
    tmem_dealloc_cg2(tmem_base, GEMM_TMEM_COLS);
  }
}

}  // namespace af
