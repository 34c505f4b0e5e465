// Segment-masked causal attention over the Unified KV Ring Buffer (step a4; Alg. 2 line 4) as UNITS that
// run on the warps of a persistent one-CTA-per-SM kernel: the last phase of layer_chain_kernel (chain.cuh), or
// attention_umma_kernel below on the per-stage path.  For head_dim 128, no window and contexts <= AU_KV_MAX; attention_kernel
// (attention.cuh) takes every other step - and, by default, the steps with a multi-row segment (there the
// units are 1.5 % slower per step; decode-only steps are 2-4 % faster with them).
//
// Why: on mma.sync a query strip walks its KV tiles one after another - ~2 us per tile step of cp.async wait + block
// barriers + a dependent chain, 9 steps for the last strip of a 276-row prefill.  Here a unit's WHOLE score matrix fits the
// tensor memory, so there is no walk:
//
//   tensor unit (segment with > 1 row, 128-row query tile, head):  Q, K, V of the visible positions -> shared memory
//       (cp.async per row: ring wrap and zero fill for free, in the 128-byte-swizzle layout UMMA reads);
//       S = Q K^T   tcgen05.mma M = 128, N <= 128 per instruction, straight into TMEM columns [0, n) as K chunks land;
//       softmax     8 warps, thread = (query row, half of the columns): pass 1 row maximum, pass 2 p = 2^(s - m) -> fp16
//                   into shared memory (over Q | K, dead by then) as the K-major A operand, row sum in fp32;
//       O = P V     tcgen05.mma with V as the MN-major B operand (the ring stores [position][head_dim]: no transpose);
//       out = O / l TMEM -> registers -> fp16 rows.
//   row unit (one-row segment, head): the decode rows.  K and V of the whole context -> shared memory, q K^T on
//       mma.sync (1 of 16 rows used; three 16-position groups per warp in flight), softmax over the context by the block,
//       p V on FMAs with fp32 probabilities (thread = two output columns x a quarter of the positions).
//
// CTA c starts with unit c and pops further units from a counter; tensor units come first (the longest).  Every reduction
// order is fixed and positions are walked in LOGICAL order: results do not depend on base_r, on the grid size, on which CTA
// ran a unit or on timing.
#pragma once
#include "attention.cuh"

namespace af {

constexpr int AU_HD = 128;                 // head_dim (two 64-element halves of 128 bytes per row)
constexpr int AU_BQ = 128;                 // query rows per tensor unit = UMMA M
constexpr int AU_KV_MAX = 352;             // positions a unit can see: S takes <= 352 of the 512 TMEM columns, O the last 128
constexpr int AU_WORKERS = 256;            // 8 load / softmax / epilogue warps
constexpr int AU_THREADS = AU_WORKERS + 32;   // + the MMA-issuing warp (also owns the TMEM allocation)
constexpr int AU_HALF_Q = AU_BQ * 128;        // bytes of one 64-element half of the Q tile
constexpr int AU_HALF_KV = AU_KV_MAX * 128;   // ... of the K (V) tile: a multiple of 1024
constexpr int AU_OFF_K = 2 * AU_HALF_Q;
constexpr int AU_OFF_V = AU_OFF_K + 2 * AU_HALF_KV;
constexpr int AU_TILE_BYTES = AU_OFF_V + 2 * AU_HALF_KV;   // 212992; P [128][<= 384] fp16 = 98304 bytes lives over Q | K
constexpr int AU_SMEM_BYTES = AU_TILE_BYTES + 1024;        // + slack to align the tiles to 1024 bytes
constexpr int AU_TMEM_COLS = 512;
constexpr int AU_O_COL = 384;
constexpr int AU_MAX_ITEMS = AF_MAX_SEGS_K + 16;           // (segment, query tile) pairs of a step
static_assert(AU_HALF_KV % 1024 == 0, "swizzle atoms are 1024 bytes");
static_assert(6 * AU_HALF_Q <= AU_OFF_V, "P overlaps V");

// MN-major B operand (V: rows = positions = K of the MMA, 64 head_dim elements = 128 bytes per row, 128-byte swizzle):
// LBO = distance between the two 64-element halves of N, SBO = 1024 B between 8-position groups, version 1, SWIZZLE_128B.
__device__ __forceinline__ uint64_t umma_smem_desc_sw128_mn(uint32_t smem_addr, uint32_t lbo_bytes) {
  uint64_t d = 0;
  d |= static_cast<uint64_t>((smem_addr & 0x3FFFF) >> 4);
  d |= static_cast<uint64_t>(lbo_bytes >> 4) << 16;
  d |= static_cast<uint64_t>(1024 >> 4) << 32;
  d |= static_cast<uint64_t>(1) << 46;
  d |= static_cast<uint64_t>(2) << 61;
  return d;
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float* v) {   // this warp's 32 lanes x 32 consecutive columns
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
      "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
      : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]), "=f"(v[8]),
        "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15]), "=f"(v[16]),
        "=f"(v[17]), "=f"(v[18]), "=f"(v[19]), "=f"(v[20]), "=f"(v[21]), "=f"(v[22]), "=f"(v[23]), "=f"(v[24]),
        "=f"(v[25]), "=f"(v[26]), "=f"(v[27]), "=f"(v[28]), "=f"(v[29]), "=f"(v[30]), "=f"(v[31])
      : "r"(taddr)
      : "memory");
}
constexpr int AU_TRACE_SLOTS = 18;   // 0 start, 1 unit lists; first two units of the CTA: 2 + 8 k + {loads issued, first chunk landed,
                                     // all landed, S done | scores, maximum, P written | probabilities, O done | V landed, unit end, -}
#define AU_STAMP(i) do { if (trace && tid == 0 && (i) < AU_TRACE_SLOTS) trace[blockIdx.x * AU_TRACE_SLOTS + (i)] = static_cast<long long>(globaltimer_ns()); } while (0)
#define AU_WORKER_BAR() asm volatile("bar.sync 1, 256;\n" ::: "memory")   // the 8 worker warps

// rows [j_lo, j_hi) (j_lo a multiple of 16) of a request's K (V) head -> the UMMA tile at `tile` (two halves of [rows][128 B],
// 128-byte swizzle); positions >= kv_end are zero-filled (V: 0 * garbage could be NaN), slot = (base + j) mod C.
// Thread = (16-byte column c = tid % 16, rows tid / 16 + 16 k): the swizzle term (c ^ j) & 7 is the same for all its rows.
__device__ __forceinline__ void au_load_rows_umma(uint8_t* tile, int half_bytes, const act_t* __restrict__ head, int base, int C,
                                                  int j_lo, int j_hi, int kv_end, int tid) {
  const int c = tid & 15;
  int j = j_lo + (tid >> 4);
  uint8_t* dst = tile + (c >> 3) * half_bytes + j * 128 + (((c & 7) ^ (j & 7)) << 4);
  int slot = base + j;
  slot = slot >= C ? slot - C : slot;
  const act_t* src = head + c * 8;
  for (; j < j_hi; j += 16) {
    cp_async16(dst, src + static_cast<size_t>(j < kv_end ? slot : 0) * AU_HD, j < kv_end);
    dst += 16 * 128;
    slot += 16;
    slot = slot >= C ? slot - C : slot;
  }
}
// the same rows as plain [row][256 B] tiles (attention.cuh's sw_off layout) for the row units
__device__ __forceinline__ void au_load_rows_plain(uint8_t* tile, const act_t* __restrict__ head, int base, int C, int n_rows, int kv_end, int tid) {
  const int c = tid & 15;
  int j = tid >> 4;
  uint8_t* dst = tile + sw_off<AU_HD>(j, c);
  int slot = base + j;
  slot = slot >= C ? slot - C : slot;
  const act_t* src = head + c * 8;
  for (; j < n_rows; j += 16) {
    cp_async16(dst, src + static_cast<size_t>(j < kv_end ? slot : 0) * AU_HD, j < kv_end);
    dst += 16 * (AU_HD * 2);
    slot += 16;
    slot = slot >= C ? slot - C : slot;
  }
}
__device__ __forceinline__ float ex2_approx(float x) {   // 2^x, one MUFU; 2^(-inf) = 0
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;\n" : "=f"(y) : "f"(x));
  return y;
}

// The step's segment table and unit lists in shared memory: they depend on the step only, so the layer chain builds them
// at kernel start (static shared memory), off the attention phase's path.
struct AuLists {
  int seg_req[AF_MAX_SEGS_K], seg_start[AF_MAX_SEGS_K], seg_len[AF_MAX_SEGS_K], seg_row0[AF_MAX_SEGS_K], seg_base[AF_MAX_SEGS_K];
  int it_seg[AU_MAX_ITEMS], it_q0[AU_MAX_ITEMS], dec_seg[AF_MAX_SEGS_K], cnt[2];
};
// Shared-memory state of a CTA's attention units besides the tiles: static in attention_umma_kernel, carved from the
// dynamic allocation (behind the tiles) in layer_chain_kernel.
struct AuAux {
  uint64_t bar_k[3], bar_v, bar_s, bar_p, bar_o;   // K chunks / V landed (256 arrivals), S done (commit), P written (256), O done (commit)
  uint64_t bar_rv;                                 // row units: V landed (bulk copies, complete_tx)
  int kvp[2];                                      // N extent of the tensor unit the MMA thread runs next, by barrier parity; 0 = no more units
  int next[2];                                     // the CTA's next unit (double-buffered across units)
  float sc[AU_KV_MAX];                             // row units: scores, then probabilities
  float mx[2][AU_BQ], sm[2][AU_BQ];                // tensor units: row maxima / sums of the two column halves
  float part[4][AU_HD];                            // row units: p V partial sums of the four position classes
  float red[16];
  __align__(16) uint8_t q[AU_HD * 2];              // row units: the query row
};
struct AuArgs {
  const act_t* q;      // [T, H*128] rotated queries
  const act_t* kv;     // ring, layer base: [2][R][H][C][128]
  act_t* out;          // [T, H*128]
  StepTables tb;
  int n_segs, H, R, C;
  float scale_log2;
  int* sched;          // {units handed out beyond the first n_cta, CTAs that have finished}: 0, 0 between launches; nullptr: unit c, c + n_cta, ..
  long long* trace;    // debug: [CTAs][AU_TRACE_SLOTS] globaltimer stamps of worker thread 0, or nullptr
};
__device__ __forceinline__ void au_init_barriers(AuAux& x) {   // one thread, before a fence_barrier_init and a block-wide barrier
  for (int i = 0; i < 3; ++i) mbar_init(&x.bar_k[i], AU_WORKERS);
  mbar_init(&x.bar_v, AU_WORKERS);
  mbar_init(&x.bar_s, 1);
  mbar_init(&x.bar_p, AU_WORKERS);
  mbar_init(&x.bar_o, 1);
  mbar_init(&x.bar_rv, 1);
}

// The MMA-issuing thread of a CTA: one pass per tensor unit of the worker warps, in their order; it learns a unit's extent
// from x.kvp (written before the workers' arrival on bar_k[0]) and leaves on the 0 the workers publish after their last unit.
__device__ __forceinline__ void au_mma_loop(AuAux& x, uint8_t* tiles, uint32_t tmem) {
  const uint32_t idesc_o = umma_idesc_f16(AU_BQ, AU_HD) | (1u << 16);   // B (= V) is MN-major
  for (uint32_t par = 0;; par ^= 1u) {
    mbar_wait(&x.bar_k[0], par);
    const int kvp = *reinterpret_cast<volatile int*>(&x.kvp[par]);
    if (kvp == 0) break;
    const int n_ch = (kvp + 127) >> 7;
    for (int ch = 0; ch < n_ch; ++ch) {      // S[:, 128 ch ..] = Q K_ch^T as soon as the chunk (and, with chunk 0, Q) has landed
      if (ch > 0) mbar_wait(&x.bar_k[ch], par);
      tc_fence_after();
      const uint32_t idesc = umma_idesc_f16(AU_BQ, static_cast<uint32_t>(min(128, kvp - ch * 128)));
#pragma unroll
      for (int ks = 0; ks < AU_HD / 16; ++ks) {
        const uint64_t a = umma_smem_desc_sw128(smem_u32(tiles + (ks >> 2) * AU_HALF_Q + (ks & 3) * 32));
        const uint64_t b = umma_smem_desc_sw128(smem_u32(tiles + AU_OFF_K + (ks >> 2) * AU_HALF_KV + ch * (128 * 128) + (ks & 3) * 32));
        umma_f16_cg1(tmem + ch * 128, a, b, idesc, ks > 0);
      }
    }
    umma_commit(&x.bar_s);
    mbar_wait(&x.bar_v, par);
    mbar_wait(&x.bar_p, par);
    tc_fence_after();
    for (int ks = 0; ks < (kvp >> 4); ++ks) {
      const uint64_t a = umma_smem_desc_sw128(smem_u32(tiles + (ks >> 2) * AU_HALF_Q + (ks & 3) * 32));   // P, 64-position chunk ks / 4
      const uint64_t b = umma_smem_desc_sw128_mn(smem_u32(tiles + AU_OFF_V + ks * 2048), AU_HALF_KV);
      umma_f16_cg1(tmem + AU_O_COL, a, b, idesc_o, ks > 0);
    }
    umma_commit(&x.bar_o);
  }
}

// Look-ahead between units.  A unit publishes the CTA's next unit (thread 0 knows it: static stride or the counter pop made at
// the unit's start) at one of its block barriers, and once its own K (tensor unit: everything) is dead it starts the q + K
// loads of a following ROW unit - one cp.async group that stays in flight across the unit boundary.
struct AuNext {
  int u_t0;       // thread 0: the next unit (other threads: ignored)
  int slot;       // x.next[slot] carries it to the block
  int n_mm, n_units;
};
__device__ __forceinline__ void au_row_issue_qk(AuAux& x, const AuLists& L, uint8_t* tiles, const AuArgs& a, int u, const AuNext& nx, int tid) {
  if (u >= nx.n_mm && u < nx.n_units) {
    const int k = (u - nx.n_mm) / a.H, h = (u - nx.n_mm) - k * a.H;
    const int seg = L.dec_seg[k];
    const int n = L.seg_start[seg] + 1;
    const act_t* kbase = a.kv + (static_cast<size_t>(0 * a.R + L.seg_req[seg]) * a.H + h) * (static_cast<size_t>(a.C) * AU_HD);
    if (tid < 16) cp_async16(x.q + tid * 16, a.q + static_cast<size_t>(L.seg_row0[seg]) * (a.H * AU_HD) + h * AU_HD + tid * 8, true);
    au_load_rows_plain(tiles, kbase, L.seg_base[seg], a.C, (n + 15) & ~15, n, tid);
  }
  cp_async_commit();   // (an empty group when nothing follows: the waits below count groups)
}

// ---- tensor unit, the 8 worker warps: (segment seg, query rows q0 .. q0 + 127, head h) ----
__device__ __forceinline__ int au_tile_unit(AuAux& x, const AuLists& L, uint8_t* tiles, uint32_t tmem, const AuArgs& a, int seg, int q0, int h,
                                            uint32_t par, const AuNext& nx, int tid, long long* trace, int ts) {
  const int warp = tid >> 5, lane = tid & 31;
  const int req = L.seg_req[seg], start = L.seg_start[seg], len = L.seg_len[seg], row0 = L.seg_row0[seg], base = L.seg_base[seg];
  const int nq = min(AU_BQ, len - q0);
  const int kv_end = start + q0 + nq;          // positions [0, kv_end) are visible to the tile's last row
  const int kvp = (kv_end + 15) & ~15;         // N extent of S = K extent of P V
  const int ldq = a.H * AU_HD;
  const size_t head_stride = static_cast<size_t>(a.C) * AU_HD;
  const act_t* kbase = a.kv + (static_cast<size_t>(0 * a.R + req) * a.H + h) * head_stride;
  const act_t* vbase = a.kv + (static_cast<size_t>(1 * a.R + req) * a.H + h) * head_stride;
  // ---- loads: Q + K[0,128) | K[128,256) | K[256,..) | V, one cp.async group each ----
  {
    const int c = tid & 15;
    const act_t* src = a.q + static_cast<size_t>(row0 + q0) * ldq + h * AU_HD + c * 8;
    uint8_t* dst = tiles + (c >> 3) * AU_HALF_Q + (tid >> 4) * 128 + (((c & 7) ^ ((tid >> 4) & 7)) << 4);
#pragma unroll
    for (int r = tid >> 4; r < AU_BQ; r += 16, dst += 16 * 128)
      cp_async16(dst, src + static_cast<size_t>(r < nq ? r : 0) * ldq, r < nq);
  }
  au_load_rows_umma(tiles + AU_OFF_K, AU_HALF_KV, kbase, base, a.C, 0, min(128, kvp), kv_end, tid);
  cp_async_commit();
  au_load_rows_umma(tiles + AU_OFF_K, AU_HALF_KV, kbase, base, a.C, 128, min(256, kvp), kv_end, tid);
  cp_async_commit();
  au_load_rows_umma(tiles + AU_OFF_K, AU_HALF_KV, kbase, base, a.C, 256, kvp, kv_end, tid);
  cp_async_commit();
  au_load_rows_umma(tiles + AU_OFF_V, AU_HALF_KV, vbase, base, a.C, 0, kvp, kv_end, tid);
  cp_async_commit();
  if (tid == 0) x.kvp[par] = kvp;
  AU_STAMP(ts + 0);
  cp_async_wait<3>(); fence_proxy_async(); mbar_arrive(&x.bar_k[0]);
  AU_STAMP(ts + 1);
  cp_async_wait<2>(); fence_proxy_async(); mbar_arrive(&x.bar_k[1]);
  cp_async_wait<1>(); fence_proxy_async(); mbar_arrive(&x.bar_k[2]);
  cp_async_wait<0>(); fence_proxy_async(); mbar_arrive(&x.bar_v);
  AU_STAMP(ts + 2);

  // ---- softmax on the TMEM rows: thread = (query row, half of the 32-column chunks) ----
  const int qd = warp & 3, hf = warp >> 2;
  const int r = qd * 32 + lane;
  const int p = start + q0 + r;                                      // this row's position
  const bool row_ok = r < nq;
  const int p_wmax = qd * 32 < nq ? start + q0 + min(qd * 32 + 31, nq - 1) : -1;   // last position any row of this warp sees
  const int n32 = (kvp + 31) >> 5, c_split = (n32 + 1) >> 1;
  const int c_lo = hf ? c_split : 0, c_hi = hf ? n32 : c_split;
  const uint32_t t_row = tmem + (static_cast<uint32_t>(qd * 32) << 16);
  float v[32];
  mbar_wait(&x.bar_s, par);
  tc_fence_after();
  AU_STAMP(ts + 3);
  float mx = -INFINITY;
  for (int c = c_lo; c < c_hi; ++c) {
    const int j0 = c * 32;
    if (j0 > p_wmax) break;                                          // above the diagonal of every row of the warp
    tmem_ld32(t_row + j0, v);
    tmem_ld_wait();
#pragma unroll
    for (int e = 0; e < 32; ++e) mx = fmaxf(mx, (j0 + e <= p) ? v[e] : -INFINITY);
  }
  x.mx[hf][r] = mx;
  if (tid == 0) x.next[nx.slot] = nx.u_t0;
  AU_WORKER_BAR();
  const int u_next = x.next[nx.slot];
  AU_STAMP(ts + 4);
  const float m = fmaxf(x.mx[0][r], x.mx[1][r]) * a.scale_log2;     // finite for a valid row: position 0 is always visible
  float sum = 0.f;
  const int p_vis = row_ok ? p : -1;                                 // rows beyond the tile see nothing
  for (int c = c_lo; c < c_hi; ++c) {
    const int j0 = c * 32;
    uint32_t pk[16];
    if (j0 <= p_wmax) {
      tmem_ld32(t_row + j0, v);
      tmem_ld_wait();
#pragma unroll
      for (int e = 0; e < 32; e += 2) {
        const float p0 = ex2_approx(j0 + e <= p_vis ? fmaf(v[e], a.scale_log2, -m) : -INFINITY);       // masked: 2^(-inf) = 0
        const float p1 = ex2_approx(j0 + e + 1 <= p_vis ? fmaf(v[e + 1], a.scale_log2, -m) : -INFINITY);
        sum += p0 + p1;
        pk[e >> 1] = pack_act(p0, p1);
      }
    } else {
#pragma unroll
      for (int e = 0; e < 16; ++e) pk[e] = 0u;
    }
    uint8_t* prow = tiles + (j0 >> 6) * AU_HALF_Q + r * 128;         // P: K-major, 64-position chunks of [128 rows][128 B]
    const int cb = (j0 & 63) >> 3;
#pragma unroll
    for (int k = 0; k < 4; ++k)
      *reinterpret_cast<uint4*>(prow + (((cb + k) ^ (r & 7)) << 4)) = make_uint4(pk[4 * k], pk[4 * k + 1], pk[4 * k + 2], pk[4 * k + 3]);
  }
  x.sm[hf][r] = sum;
  fence_proxy_async();
  tc_fence_before();
  mbar_arrive(&x.bar_p);
  AU_WORKER_BAR();
  AU_STAMP(ts + 5);
  const float inv = 1.f / (x.sm[0][r] + x.sm[1][r]);
  // ---- out = O / l: this thread's row, 64 of the 128 columns ----
  mbar_wait(&x.bar_o, par);
  tc_fence_after();
  AU_STAMP(ts + 6);
  au_row_issue_qk(x, L, tiles, a, u_next, nx, tid);   // Q, K, P and V are dead: a following row unit's loads fly during the epilogue
  act_t* dst = a.out + static_cast<size_t>(row0 + q0 + (row_ok ? r : 0)) * ldq + h * AU_HD + hf * 64;
#pragma unroll
  for (int cc = 0; cc < 2; ++cc) {
    tmem_ld32(t_row + AU_O_COL + hf * 64 + cc * 32, v);
    tmem_ld_wait();
    if (row_ok) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        *reinterpret_cast<uint4*>(dst + cc * 32 + k * 8) =
            make_uint4(pack_act(v[8 * k] * inv, v[8 * k + 1] * inv), pack_act(v[8 * k + 2] * inv, v[8 * k + 3] * inv),
                       pack_act(v[8 * k + 4] * inv, v[8 * k + 5] * inv), pack_act(v[8 * k + 6] * inv, v[8 * k + 7] * inv));
    }
  }
  tc_fence_before();
  AU_STAMP(ts + 7);
  return u_next;
}

// ---- row unit, the 8 worker warps: (one-row segment seg, head h) - a decode row against its whole context ----
__device__ __forceinline__ int au_row_unit(AuAux& x, const AuLists& L, uint8_t* tiles, const AuArgs& a, int seg, int h, bool qk_in_flight,
                                           uint32_t rpar, const AuNext& nx, int tid, long long* trace, int ts) {
  const int warp = tid >> 5, lane = tid & 31;
  const int req = L.seg_req[seg], start = L.seg_start[seg], row0 = L.seg_row0[seg], base = L.seg_base[seg];
  const int n = start + 1;                      // the row sees positions [0, start]
  const int n16 = (n + 15) & ~15;
  const int ldq = a.H * AU_HD;
  const size_t head_stride = static_cast<size_t>(a.C) * AU_HD;
  const act_t* kbase = a.kv + (static_cast<size_t>(0 * a.R + req) * a.H + h) * head_stride;
  const act_t* vbase = a.kv + (static_cast<size_t>(1 * a.R + req) * a.H + h) * head_stride;
  uint8_t* sK = tiles;
  uint8_t* sV = tiles + AU_KV_MAX * (AU_HD * 2);
  if (!qk_in_flight) {     // (else: the previous unit started them, one group)
    if (tid < 16) cp_async16(x.q + tid * 16, a.q + static_cast<size_t>(row0) * ldq + h * AU_HD + tid * 8, true);
    au_load_rows_plain(sK, kbase, base, a.C, n16, n, tid);
    cp_async_commit();
  }
  // V: plain [position][256 B] rows, read row by row in p V - no swizzle needed, so the ring range goes in as one or two
  // bulk copies (the wrap) instead of 4.6 k cp.async, and the LSU queue is K's alone
  if (tid == 0) {
    fence_proxy_async();      // the previous unit's generic reads of this buffer (ordered by the block barrier) before the async writes
    const int n1 = min(n, a.C - base);
    mbar_arrive_expect_tx(&x.bar_rv, static_cast<uint32_t>(n) * (AU_HD * 2));
    bulk_load_1d(sV, vbase + static_cast<size_t>(base) * AU_HD, static_cast<uint32_t>(n1) * (AU_HD * 2), &x.bar_rv);
    if (n1 < n) bulk_load_1d(sV + n1 * (AU_HD * 2), vbase, static_cast<uint32_t>(n - n1) * (AU_HD * 2), &x.bar_rv);
  }
  AU_STAMP(ts + 0);
  cp_async_wait<0>();
  AU_WORKER_BAR();
  AU_STAMP(ts + 1);
  // ---- scores: q K^T on mma.sync, the query in row 0 of the A fragment; warp w takes 16-position groups w, w + 8, .. ----
  {
    const int g = lane >> 2, t = lane & 3;
    uint32_t qa[AU_HD / 16][4];
#pragma unroll
    for (int kk = 0; kk < AU_HD / 16; ++kk) {
      qa[kk][0] = g == 0 ? *reinterpret_cast<const uint32_t*>(x.q + (kk * 16 + 2 * t) * 2) : 0u;
      qa[kk][2] = g == 0 ? *reinterpret_cast<const uint32_t*>(x.q + (kk * 16 + 8 + 2 * t) * 2) : 0u;
      qa[kk][1] = 0u; qa[kk][3] = 0u;
    }
    // the warp's (up to) three groups in one pass: three independent accumulator chains instead of three serial ones
    float s0[3][4], s1[3][4];
#pragma unroll
    for (int gi = 0; gi < 3; ++gi)
#pragma unroll
      for (int e = 0; e < 4; ++e) { s0[gi][e] = 0.f; s1[gi][e] = 0.f; }
#pragma unroll
    for (int kk = 0; kk < AU_HD / 16; ++kk) {
#pragma unroll
      for (int gi = 0; gi < 3; ++gi) {
        const int j0 = (warp + 8 * gi) * 16;
        if (j0 < n16) {                      // warp-uniform
          uint32_t b0, b1, b2, b3;
          const int r = j0 + (lane & 7) + (lane >> 4) * 8;
          const int c = kk * 2 + ((lane >> 3) & 1);
          ldsm_x4(smem_u32(sK + sw_off<AU_HD>(r, c)), b0, b1, b2, b3);
          mma_f16_16816(s0[gi], qa[kk], b0, b1);
          mma_f16_16816(s1[gi], qa[kk], b2, b3);
        }
      }
    }
#pragma unroll
    for (int gi = 0; gi < 3; ++gi) {
      const int j = (warp + 8 * gi) * 16 + 2 * t;
      if (g == 0 && (warp + 8 * gi) * 16 < n16) {
        x.sc[j] = j < n ? s0[gi][0] * a.scale_log2 : -INFINITY;
        x.sc[j + 1] = j + 1 < n ? s0[gi][1] * a.scale_log2 : -INFINITY;
        x.sc[j + 8] = j + 8 < n ? s1[gi][0] * a.scale_log2 : -INFINITY;
        x.sc[j + 9] = j + 9 < n ? s1[gi][1] * a.scale_log2 : -INFINITY;
      }
    }
  }
  if (tid == 0) x.next[nx.slot] = nx.u_t0;
  AU_WORKER_BAR();
  AU_STAMP(ts + 3);
  const int u_next = x.next[nx.slot];
  au_row_issue_qk(x, L, tiles, a, u_next, nx, tid);   // this unit's q and K are dead: a following row unit's fly during the softmax and p V
  // ---- softmax over the context: thread t holds positions t and t + 256 ----
  const float x0 = tid < n16 ? x.sc[tid] : -INFINITY;
  const float x1 = tid + AU_WORKERS < n16 ? x.sc[tid + AU_WORKERS] : -INFINITY;
  float mx = fmaxf(x0, x1);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) x.red[warp] = mx;
  AU_WORKER_BAR();
  AU_STAMP(ts + 4);
  float m = x.red[0];
#pragma unroll
  for (int i = 1; i < 8; ++i) m = fmaxf(m, x.red[i]);
  const float p0 = ex2_approx(x0 - m), p1 = ex2_approx(x1 - m);   // 2^(-inf) = 0 beyond the context
  if (tid < n16) x.sc[tid] = p0;
  if (tid + AU_WORKERS < n16) x.sc[tid + AU_WORKERS] = p1;
  float sum = p0 + p1;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if (lane == 0) x.red[8 + warp] = sum;
  mbar_wait(&x.bar_rv, rpar);   // V has landed
  AU_WORKER_BAR();
  AU_STAMP(ts + 5);
  float l = x.red[8];
#pragma unroll
  for (int i = 1; i < 8; ++i) l += x.red[8 + i];
  // ---- out = p V / l: thread = (column pair cp, position class j mod 4), classes added up in order ----
  {
    const int cp = tid & 63, sub = tid >> 6;
    float a0 = 0.f, a1 = 0.f;
    int j = sub;
    for (; j + 12 < n; j += 16) {      // four positions in flight (loads first), added in position order
      float pj[4];
      float2 vv[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        pj[i] = x.sc[j + 4 * i];
        vv[i] = __half22float2(*reinterpret_cast<const __half2*>(sV + (j + 4 * i) * (AU_HD * 2) + cp * 4));
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) { a0 = fmaf(pj[i], vv[i].x, a0); a1 = fmaf(pj[i], vv[i].y, a1); }
    }
    for (; j < n; j += 4) {
      const float pj = x.sc[j];
      const float2 vv = __half22float2(*reinterpret_cast<const __half2*>(sV + j * (AU_HD * 2) + cp * 4));
      a0 = fmaf(pj, vv.x, a0); a1 = fmaf(pj, vv.y, a1);
    }
    x.part[sub][2 * cp] = a0; x.part[sub][2 * cp + 1] = a1;
  }
  AU_WORKER_BAR();
  if (tid < 64) {
    const float inv = 1.f / l;
    const float o0 = ((x.part[0][2 * tid] + x.part[1][2 * tid]) + x.part[2][2 * tid]) + x.part[3][2 * tid];
    const float o1 = ((x.part[0][2 * tid + 1] + x.part[1][2 * tid + 1]) + x.part[2][2 * tid + 1]) + x.part[3][2 * tid + 1];
    *reinterpret_cast<uint32_t*>(a.out + static_cast<size_t>(row0) * ldq + h * AU_HD + 2 * tid) = pack_act(o0 * inv, o1 * inv);
  }
  AU_STAMP(ts + 7);
  return u_next;
}

// Segment table -> unit lists, by `nthr` threads (a multiple of 32) that meet at named barrier `bar_id`: (segment, query
// tile) of every multi-row segment, longest context first, and the one-row segments.
__device__ __forceinline__ void au_build_lists(AuLists& L, const StepTables& tb, int n_segs, int tid) {
  for (int s = tid; s < n_segs; s += AU_WORKERS) {
    L.seg_req[s] = tb.seg_req[s]; L.seg_start[s] = tb.seg_start[s]; L.seg_len[s] = tb.seg_len[s];
    L.seg_row0[s] = tb.seg_row0[s]; L.seg_base[s] = tb.seg_base[s];
  }
  AU_WORKER_BAR();
  if (tid == 0) {
    int n_it = 0, n_dec = 0;
    for (int s = 0; s < n_segs; ++s) {
      const int len = L.seg_len[s];
      if (len == 1) { L.dec_seg[n_dec++] = s; continue; }
      for (int q0 = ((len - 1) / AU_BQ) * AU_BQ; q0 >= 0 && n_it < AU_MAX_ITEMS; q0 -= AU_BQ) { L.it_seg[n_it] = s; L.it_q0[n_it] = q0; ++n_it; }
    }
    L.cnt[0] = n_it; L.cnt[1] = n_dec;
  }
  AU_WORKER_BAR();
}

// The worker warps' side of a CTA (tid 0..255), lists built: this CTA's units.  Tensor units come first (the longest).
// With a.sched the CTA starts with unit `cta` and pops every further one from a counter - at the START of the current
// unit, so the atomic's round trip is hidden; otherwise it takes units cta, cta + n_cta, ...  Which CTA runs a unit does not
// change its result.
__device__ __forceinline__ void au_workers(AuAux& x, const AuLists& L, uint8_t* tiles, uint32_t tmem, const AuArgs& a, int cta, int n_cta, int tid) {
  long long* trace = a.trace;
  AU_STAMP(1);
  const int n_mm = L.cnt[0] * a.H, n_units = n_mm + L.cnt[1] * a.H;
  int n_done = 0;
  uint32_t par = 0;   // phase parity of the tensor units' mbarriers (each completes once per tensor unit)
  uint32_t rpar = 0;  // ... of the row units' V barrier
  int u = cta;
  bool qk_in_flight = false;   // the current (row) unit's q + K loads were started by the previous unit
  while (u < n_units) {
    AuNext nx;
    nx.u_t0 = u + n_cta; nx.slot = n_done & 1; nx.n_mm = n_mm; nx.n_units = n_units;
    if (a.sched && tid == 0) nx.u_t0 = n_cta + atomicAdd(&a.sched[0], 1);
    int u_next;
    if (u < n_mm) {
      const int it = u / a.H;
      u_next = au_tile_unit(x, L, tiles, tmem, a, L.it_seg[it], L.it_q0[it], u - it * a.H, par, nx, tid, trace, 2 + 8 * n_done);
      par ^= 1u;
    } else {
      const int k = (u - n_mm) / a.H;
      u_next = au_row_unit(x, L, tiles, a, L.dec_seg[k], (u - n_mm) - k * a.H, qk_in_flight, rpar, nx, tid, trace, 2 + 8 * n_done);
      rpar ^= 1u;
    }
    AU_WORKER_BAR();   // the unit's shared-memory reads (V, the partial sums) are over before the next unit's loads
    qk_in_flight = u_next >= n_mm && u_next < n_units;
    u = u_next;
    ++n_done;
  }
  if (tid == 0) x.kvp[par] = 0;   // tell the MMA thread there is no further tensor unit
  mbar_arrive(&x.bar_k[0]);
  if (a.sched && tid == 0 && atomicAdd(&a.sched[1], 1) == n_cta - 1) { a.sched[0] = 0; a.sched[1] = 0; }   // the last CTA out resets both
}

// The kernel of its own: used where the layer chain does not run (the per-stage path).  One CTA per SM.
__global__ void __launch_bounds__(AU_THREADS, 1)
attention_umma_kernel(const AuArgs a) {
  extern __shared__ uint8_t au_smem_raw[];
  uint8_t* tiles = au_smem_raw + ((1024u - (smem_u32(au_smem_raw) & 1023u)) & 1023u);
  __shared__ AuAux x;
  __shared__ AuLists lists;
  __shared__ uint32_t s_tmem;
  const int tid = threadIdx.x, warp = tid >> 5;
  if (warp == 8) tmem_alloc(&s_tmem, AU_TMEM_COLS);
  if (tid == 0) {
    au_init_barriers(x);
    fence_barrier_init();
  }
  pdl_wait();
  pdl_launch_dependents();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;
  if (warp < 8) {
    long long* trace = a.trace;
    AU_STAMP(0);
    au_build_lists(lists, a.tb, a.n_segs, tid);
    au_workers(x, lists, tiles, tmem, a, blockIdx.x, gridDim.x, tid);
  }
  else if (tid == AU_WORKERS) au_mma_loop(x, tiles, tmem);
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc(tmem, AU_TMEM_COLS);
}

}  // namespace af
