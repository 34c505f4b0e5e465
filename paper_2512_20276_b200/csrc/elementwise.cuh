// Row-wise kernels of the packed forward: segment-table ingest (a0), residual + RMSNorm (a5/a8 + a1/a6),
// RoPE + ring append (a3), logits-row gather + final norm (a10), RoPE table.  SURVEY.md 8(a); Alg. 2 lines 1 and 3
// (P:180-182).  SiLU*mul (a7) is an epilogue of the GEMM kernel (gemm_tcgen05.cuh).
#pragma once
#include "attention.cuh"

namespace af {

struct SegTableArg {  // the host segment table, passed by value as a kernel parameter (no staging copy)
  int n_segs;
  int R, C;
  int req[AF_MAX_SEGS_K], start[AF_MAX_SEGS_K], len[AF_MAX_SEGS_K], base[AF_MAX_SEGS_K];
};

// a0: every packed row i -> (req, pos = start_pos + i - row0(seg), slot = req*C + (base_r + pos) mod C), plus the
// per-segment arrays and the attention work list.  One block; all integer, bit-exact by construction (P:208
// "precomputed physical address").
__device__ __forceinline__ void rowmap_body(const SegTableArg& st, StepTables tb, int* n_items_out) {
  __shared__ int row0[AF_MAX_SEGS_K + 1], item0[AF_MAX_SEGS_K + 1];
  if (threadIdx.x == 0) {
    int r = 0, it = 0;
    for (int s = 0; s < st.n_segs; ++s) {
      row0[s] = r; item0[s] = it;
      r += st.len[s];
      it += (st.len[s] + ATT_BQ - 1) / ATT_BQ;
    }
    row0[st.n_segs] = r; item0[st.n_segs] = it;
    *n_items_out = it;
  }
  __syncthreads();
  for (int s = threadIdx.x; s < st.n_segs; s += blockDim.x) {
    tb.seg_req[s] = st.req[s]; tb.seg_start[s] = st.start[s]; tb.seg_len[s] = st.len[s];
    tb.seg_row0[s] = row0[s]; tb.seg_base[s] = st.base[s];
    const int n_it = item0[s + 1] - item0[s];
    for (int k = 0; k < n_it; ++k) { tb.item_tmp[2 * (item0[s] + k)] = s; tb.item_tmp[2 * (item0[s] + k) + 1] = k * ATT_BQ; }
  }
  __syncthreads();
  // attention work list, heaviest first (cost = query warps x visible KV tiles): the grid is (heads, items), so the
  // block scheduler hands every SM one heavy item before the light ones - the kernel is one wave, placement is all
  const int n_items = item0[st.n_segs];
  auto cost = [&](int it) {
    const int s = tb.item_tmp[2 * it], q0 = tb.item_tmp[2 * it + 1];
    const int nq = min(ATT_BQ, st.len[s] - q0);
    return ((nq + 15) / 16) * ((st.start[s] + q0 + nq + ATT_BKV - 1) / ATT_BKV);
  };
  for (int it = threadIdx.x; it < n_items; it += blockDim.x) {
    const int c = cost(it);
    int rank = 0;
    for (int j = 0; j < n_items; ++j) {
      const int cj = cost(j);
      rank += (cj > c || (cj == c && j < it)) ? 1 : 0;
    }
    tb.item_seg[rank] = tb.item_tmp[2 * it]; tb.item_q0[rank] = tb.item_tmp[2 * it + 1];
  }
  const int T = row0[st.n_segs];
  for (int i = threadIdx.x; i < T; i += blockDim.x) {
    int s = 0;
    while (i >= row0[s + 1]) ++s;
    const int pos = st.start[s] + (i - row0[s]);
    tb.row_req[i] = st.req[s];
    tb.row_pos[i] = pos;
    tb.row_slot[i] = st.req[s] * st.C + (st.base[s] + pos) % st.C;
  }
}

__global__ void rowmap_kernel(const SegTableArg st, StepTables tb, int* n_items_out) { rowmap_body(st, tb, n_items_out); }

// The same ingest from a segment table that lives on the DEVICE (written by loop_advance_kernel below).
__global__ void rowmap_dev_kernel(const SegTableArg* __restrict__ st_dev, StepTables tb, int* n_items_out) {
  __shared__ SegTableArg st;
  for (int i = threadIdx.x; i < static_cast<int>(sizeof(SegTableArg) / sizeof(int)); i += blockDim.x)
    reinterpret_cast<int*>(&st)[i] = reinterpret_cast<const int*>(st_dev)[i];
  __syncthreads();
  rowmap_body(st, tb, n_items_out);
}

// ---------------------------------------------------------------------------------------------------------------------
// f1: Algorithm 1's pipeline state on the device.  Step t packs the prefill of frame t (region t mod R,
// recycled first: base <- (base + len) mod C, len <- 0, the same rule as af_ring_reset_slot(new_base = -1)) with decode
// stage s = 1..min(t, K-1) of frame t - s (region (t - s) mod R) at position len[region] = L_P + s - 1.  All integer.
struct LoopState {
  int t;                        // steps completed
  int L_P, K, R, C;
  int frame_id;                 // frame whose K tokens sit in frame_tok (-1 before the first frame completes)
  int frame_tok[AF_MAX_SEGS_K];                  // [K] tokens of the last completed frame (directly after frame_id)
  int base[AF_MAX_SEGS_K], len[AF_MAX_SEGS_K];   // per region (R <= AF_MAX_SEGS)
  int seq[AF_MAX_SEGS_K * AF_MAX_SEGS_K];        // A_sequences [R][K] (Alg. 1 l.9), token of stage s of the frame in region r
};

__global__ void loop_advance_kernel(LoopState* __restrict__ ls, SegTableArg* __restrict__ st) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int t = ls->t, R = ls->R, C = ls->C, K = ls->K;
  const int r0 = t % R;
  ls->base[r0] = (ls->base[r0] + ls->len[r0]) % C;
  ls->len[r0] = 0;
  const int n_dec = t < K - 1 ? t : K - 1;
  st->n_segs = 1 + n_dec; st->R = R; st->C = C;
  for (int s = 0; s <= n_dec; ++s) {
    const int r = (t - s) % R;
    const int n = s == 0 ? ls->L_P : 1;
    st->req[s] = r; st->start[s] = ls->len[r]; st->len[s] = n; st->base[s] = ls->base[r];
    ls->len[r] += n;             // a9: the commit is a relabelling
  }
}

// End of step t: tok[s] is the token of stage s (prediction row s of the step).  Record it in A_sequences; the frame that
// just took stage K-1 is complete: publish its K tokens.  Then t <- t + 1.
__global__ void loop_commit_kernel(LoopState* __restrict__ ls, const int* __restrict__ tok) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int t = ls->t, R = ls->R, K = ls->K;
  const int n_dec = t < K - 1 ? t : K - 1;
  for (int s = 0; s <= n_dec; ++s) ls->seq[((t - s) % R) * K + s] = tok[s];
  if (n_dec == K - 1) {
    const int r = (t - (K - 1)) % R;
    for (int s = 0; s < K; ++s) ls->frame_tok[s] = ls->seq[r * K + s];
    ls->frame_id = t - (K - 1);
  }
  ls->t = t + 1;
}

// bf16 embeddings -> fp32 residual stream
__global__ void embed_to_residual_kernel(const __nv_bfloat16* __restrict__ e, float* __restrict__ x, size_t n) {
  pdl_wait();
  pdl_launch_dependents();
  const size_t i = (static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x) * 4;
  if (i + 3 < n) {
    const uint2 raw = *reinterpret_cast<const uint2*>(e + i);
    const __nv_bfloat162 a = *reinterpret_cast<const __nv_bfloat162*>(&raw.x);
    const __nv_bfloat162 b = *reinterpret_cast<const __nv_bfloat162*>(&raw.y);
    *reinterpret_cast<float4*>(x + i) =
        make_float4(__low2float(a), __high2float(a), __low2float(b), __high2float(b));
  } else {
    for (size_t k = i; k < n; ++k) x[k] = __bfloat162float(e[k]);
  }
}

__device__ __forceinline__ float block_sum(float v, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) red[w] = v;
  __syncthreads();
  const int nw = blockDim.x >> 5;
  float t = (l < nw) ? red[l] : 0.f;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  __syncthreads();
  return t;
}

// a5/a8 residual + a1/a6 RMSNorm in one pass (and a10's norm when rows != nullptr), one block per row:
//   x[i,:] += sum_s parts[s][i,:]      the split-K partials (fp16 slabs, summed in fp32) of the preceding O / down
//                                      projection, in split order
//   y[i,:]  = fp16( x[src,:] * g / sqrt(mean(x^2) + eps) )          (skipped when g == nullptr: reduce only)
__device__ __forceinline__ void residual_norm_row(float* __restrict__ x, const act_t* __restrict__ parts, int n_parts,
                                                  long long part_stride, const __nv_bfloat16* __restrict__ g,
                                                  act_t* __restrict__ y, int i, int src, int D, float eps) {
  __shared__ float red[32];
  float* xr = x + static_cast<size_t>(src) * D;
  float ss = 0.f;
#pragma unroll 2
  for (int c = threadIdx.x * 4; c < D; c += blockDim.x * 4) {
    float4 v = *reinterpret_cast<const float4*>(xr + c);
    if (n_parts > 0) {
      const act_t* pr = parts + static_cast<size_t>(src) * D + c;
      for (int s = 0; s < n_parts; ++s) {
        const uint2 raw = __ldcg(reinterpret_cast<const uint2*>(pr + s * part_stride));
        const float2 a0 = __half22float2(*reinterpret_cast<const __half2*>(&raw.x));
        const float2 a1 = __half22float2(*reinterpret_cast<const __half2*>(&raw.y));
        v.x += a0.x; v.y += a0.y; v.z += a1.x; v.w += a1.y;
      }
      *reinterpret_cast<float4*>(xr + c) = v;
    }
    ss += v.x * v.x + v.y * v.y + v.z * v.z + v.w * v.w;
  }
  if (!g) return;
  ss = block_sum(ss, red);
  const float inv = rsqrtf(ss / D + eps);
  act_t* yr = y + static_cast<size_t>(i) * D;
  for (int c = threadIdx.x * 4; c < D; c += blockDim.x * 4) {
    const float4 v = *reinterpret_cast<const float4*>(xr + c);   // this thread's own writes (same addresses)
    const uint2 graw = *reinterpret_cast<const uint2*>(g + c);
    const __nv_bfloat162 g0 = *reinterpret_cast<const __nv_bfloat162*>(&graw.x);
    const __nv_bfloat162 g1 = *reinterpret_cast<const __nv_bfloat162*>(&graw.y);
    uint2 o;
    o.x = pack_act(v.x * inv * __low2float(g0), v.y * inv * __high2float(g0));
    o.y = pack_act(v.z * inv * __low2float(g1), v.w * inv * __high2float(g1));
    *reinterpret_cast<uint2*>(yr + c) = o;
  }
}

__global__ void __launch_bounds__(512, 2)
residual_norm_kernel(float* __restrict__ x, const act_t* __restrict__ parts, int n_parts, long long part_stride,
                     const __nv_bfloat16* __restrict__ g, act_t* __restrict__ y, int D, float eps) {
  pdl_wait();
  pdl_launch_dependents();
  residual_norm_row(x, parts, n_parts, part_stride, g, y, blockIdx.x, blockIdx.x, D, eps);
}

struct RowListArg { int rows[256]; };  // a10: the caller's row list, passed by value (no staging copy)

// a10: y[i,:] = fp16( RMSNorm(hidden[rows[i],:]; g_final) ), the input of the LM-head GEMM
__global__ void __launch_bounds__(512, 2)
gather_norm_kernel(const RowListArg rl, const float* __restrict__ x, const __nv_bfloat16* __restrict__ g,
                   act_t* __restrict__ y, int D, float eps) {
  pdl_wait();
  pdl_launch_dependents();
  residual_norm_row(const_cast<float*>(x), nullptr, 0, 0, g, y, blockIdx.x, rl.rows[blockIdx.x], D, eps);
}

// a3 FusedRoPEAndWriteKV (Alg. 2 l.3): rotate q and k of every (row, head) at the row's logical
// position in its own request (rotate-half pairing, table built in fp64), write q to the query buffer and
// k (rotated), v straight to the row's ring slot.  One block per row, 8 elements (16 bytes) per thread-iteration.
__global__ void __launch_bounds__(512, 2)
rope_append_kernel(const act_t* __restrict__ qkv,   // [T, 3*H*hd]  (q | k | v)
                   act_t* __restrict__ q_out,       // [T, H*hd]
                   act_t* __restrict__ kv_layer,    // [2][R][H][C][hd]
                   const float2* __restrict__ rope_tab,     // [C][hd/2] (cos, sin)
                   StepTables tb, int H, int hd, int R, int C) {
  pdl_wait();
  pdl_launch_dependents();
  const int i = blockIdx.x;
  const int pos = tb.row_pos[i], gslot = tb.row_slot[i];
  const int req = gslot / C, slot = gslot - req * C;
  const int D = H * hd, half = hd >> 1;
  const act_t* src = qkv + static_cast<size_t>(i) * 3 * D;
  const float2* tab = rope_tab + static_cast<size_t>(pos) * half;
  const int per_head = half / 8;  // 16-byte groups of the low half of a head
  // q and k: thread handles 8 low-half elements c..c+7 and their partners c+half..
  for (int w = threadIdx.x; w < 2 * H * per_head; w += blockDim.x) {
    const int which = w / (H * per_head);           // 0 = q, 1 = k
    const int rem = w - which * H * per_head;
    const int h = rem / per_head, c = (rem - h * per_head) * 8;
    const act_t* s = src + which * D + h * hd + c;
    const uint4 lo_raw = *reinterpret_cast<const uint4*>(s);
    const uint4 hi_raw = *reinterpret_cast<const uint4*>(s + half);
    const act_t* lo = reinterpret_cast<const act_t*>(&lo_raw);
    const act_t* hi = reinterpret_cast<const act_t*>(&hi_raw);
    uint4 out_lo, out_hi;
    uint32_t* ol = reinterpret_cast<uint32_t*>(&out_lo);
    uint32_t* oh = reinterpret_cast<uint32_t*>(&out_hi);
#pragma unroll
    for (int e = 0; e < 8; e += 2) {
      const float2 cs0 = tab[c + e], cs1 = tab[c + e + 1];
      const float l0 = act2f(lo[e]), l1 = act2f(lo[e + 1]);
      const float h0 = act2f(hi[e]), h1 = act2f(hi[e + 1]);
      ol[e >> 1] = pack_act(l0 * cs0.x - h0 * cs0.y, l1 * cs1.x - h1 * cs1.y);
      oh[e >> 1] = pack_act(h0 * cs0.x + l0 * cs0.y, h1 * cs1.x + l1 * cs1.y);
    }
    act_t* dst = (which == 0)
        ? q_out + static_cast<size_t>(i) * D + h * hd + c
        : kv_layer + ((static_cast<size_t>(0 * R + req) * H + h) * C + slot) * hd + c;
    *reinterpret_cast<uint4*>(dst) = out_lo;
    *reinterpret_cast<uint4*>(dst + half) = out_hi;
  }
  // v: plain copy into the ring
  for (int w = threadIdx.x; w < D / 8; w += blockDim.x) {
    const int h = (w * 8) / hd, c = (w * 8) - h * hd;
    const uint4 v = *reinterpret_cast<const uint4*>(src + 2 * D + w * 8);
    *reinterpret_cast<uint4*>(kv_layer + ((static_cast<size_t>(1 * R + req) * H + h) * C + slot) * hd + c) = v;
  }
}

// Load-time weight preparation: bf16 -> fp16, exact for finite |w| in [2^-14, 65504] (8 elements per thread).
__global__ void convert_bf16_to_fp16_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, size_t n_vec) {
  const size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n_vec) return;
  uint4 v = src[i];
  v.x = bf16x2_to_f16x2(v.x); v.y = bf16x2_to_f16x2(v.y); v.z = bf16x2_to_f16x2(v.z); v.w = bf16x2_to_f16x2(v.w);
  dst[i] = v;
}

// Load-time preparation of gate | up (af_prepare_gate_up): dst row t*128 + q*32 + half*16 + i = fp16 of row
// 64t + 16q + i of gate (half 0) or up (half 1); zero rows past F.  8 elements per thread.
__global__ void interleave_gate_up_kernel(const uint4* __restrict__ gate, const uint4* __restrict__ up, uint4* __restrict__ dst,
                                          int F, int vec_per_row, size_t n_vec) {
  const size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n_vec) return;
  const int row = static_cast<int>(i / vec_per_row), c = static_cast<int>(i - static_cast<size_t>(row) * vec_per_row);
  const int t = row >> 7, q = (row >> 5) & 3, half = (row >> 4) & 1, f = t * 64 + q * 16 + (row & 15);
  uint4 v = make_uint4(0u, 0u, 0u, 0u);
  if (f < F) {
    v = (half ? up : gate)[static_cast<size_t>(f) * vec_per_row + c];
    v.x = bf16x2_to_f16x2(v.x); v.y = bf16x2_to_f16x2(v.y); v.z = bf16x2_to_f16x2(v.z); v.w = bf16x2_to_f16x2(v.w);
  }
  dst[i] = v;
}

// The same row order for one-byte elements (af_prepare_gate_up_fp8: E4M3 codes are copied, not converted): 16 codes per thread.
__global__ void interleave_gate_up_bytes_kernel(const uint4* __restrict__ gate, const uint4* __restrict__ up, uint4* __restrict__ dst,
                                                int F, int vec_per_row, size_t n_vec) {
  const size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n_vec) return;
  const int row = static_cast<int>(i / vec_per_row), c = static_cast<int>(i - static_cast<size_t>(row) * vec_per_row);
  const int t = row >> 7, q = (row >> 5) & 3, half = (row >> 4) & 1, f = t * 64 + q * 16 + (row & 15);
  dst[i] = f < F ? (half ? up : gate)[static_cast<size_t>(f) * vec_per_row + c] : make_uint4(0u, 0u, 0u, 0u);
}

// f1: ArgMax over one logits row per block (Alg. 1 l.5/l.8).  (value, index) pairs are reduced with "greater value, or
// equal value and lower index, wins", which is associative and commutative, so the result does not depend on the
// reduction order: the lowest index of the maximum.  NaNs lose every comparison.
__global__ void __launch_bounds__(256)
argmax_rows_kernel(const float* __restrict__ logits, int vocab, int* __restrict__ tokens_out) {
  __shared__ float s_v[8];
  __shared__ int s_i[8];
  const float* row = logits + static_cast<size_t>(blockIdx.x) * vocab;
  float best = -INFINITY;
  int best_i = 0x7fffffff;
  for (int v = threadIdx.x; v < vocab; v += blockDim.x) {
    const float x = row[v];
    if (x > best || (x == best && v < best_i)) { best = x; best_i = v; }
  }
  auto better = [](float a, int ai, float b, int bi) { return a > b || (a == b && ai < bi); };
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, best, o);
    const int oi = __shfl_xor_sync(0xffffffffu, best_i, o);
    if (better(ov, oi, best, best_i)) { best = ov; best_i = oi; }
  }
  if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = best; s_i[threadIdx.x >> 5] = best_i; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < static_cast<int>(blockDim.x >> 5); ++w)
      if (better(s_v[w], s_i[w], best, best_i)) { best = s_v[w]; best_i = s_i[w]; }
    tokens_out[blockIdx.x] = best_i == 0x7fffffff ? 0 : best_i;
  }
}

// f1: embeds_out[i, :] = table[tokens[i], :] (16 bytes per thread-iteration); a token outside [0, vocab) gives zeros
__global__ void embed_rows_kernel(const uint4* __restrict__ table, int vocab, int vec_per_row,
                                  const int* __restrict__ tokens, uint4* __restrict__ out) {
  const int tok = tokens[blockIdx.x];
  const bool ok = tok >= 0 && tok < vocab;
  for (int c = threadIdx.x; c < vec_per_row; c += blockDim.x)
    out[static_cast<size_t>(blockIdx.x) * vec_per_row + c] =
        ok ? table[static_cast<size_t>(tok) * vec_per_row + c] : make_uint4(0u, 0u, 0u, 0u);
}

// RoPE table in fp64: tab[pos][c] = (cos, sin)(pos * theta^(-2c/hd))
__global__ void rope_table_kernel(float2* tab, int C, int hd, double theta) {
  const int half = hd / 2;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= C * half) return;
  const int pos = idx / half, c = idx - pos * half;
  const double f = exp2(-2.0 * c / hd * log2(theta));
  const double a = pos * f;
  tab[idx] = make_float2(static_cast<float>(cos(a)), static_cast<float>(sin(a)));
}

}  // namespace af
