// Segment-masked causal attention over the Unified KV Ring Buffer (step a4; Alg. 2 line 4, P:183,
// P:194-200).  Each work item is (segment, 64-row query tile) x head.  The tile's rows attend to positions
// 0..own position of THEIR OWN request only; K/V rows are gathered from the ring at slot (base_r + j) mod C
// (wrap included) with 128-bit cp.async loads into XOR-swizzled shared memory, S = QK^T and O = PV run on
// mma.sync.m16n8k16 (fp16 in, fp32 accumulate), and the online softmax reduces across the 4 lanes that share a row
// with warp shuffles.  KV tiles are walked in LOGICAL position order, so results do not depend on base_r.
#pragma once
#include "ptx.cuh"

namespace af {

constexpr int ATT_BQ = 32;       // query rows per work item: two 16-row strips, each taken by TWO warps on alternate KV tiles
constexpr int ATT_BKV = 32;
#ifndef AF_ATT_STAGES
#define AF_ATT_STAGES 3
#endif
constexpr int ATT_STAGES = AF_ATT_STAGES;   // K/V tiles in flight (cp.async groups)
__host__ __device__ constexpr int att_smem_bytes(int hd) { return (ATT_BQ + 2 * ATT_STAGES * ATT_BKV) * hd * 2; }
constexpr int ATT_THREADS = 128;

struct StepTables {      // device arrays written by rowmap_kernel (elementwise.cuh), one set per ring
  int* seg_req;          // [n_segs]
  int* seg_start;        // [n_segs] start_pos
  int* seg_len;          // [n_segs]
  int* seg_row0;         // [n_segs] first packed row
  int* seg_base;         // [n_segs] base_r of the segment's region
  int* row_req;          // [T]
  int* row_pos;          // [T]
  int* row_slot;         // [T] global slot id req*C + (base+pos) mod C
  int* item_seg;         // [n_items] attention work items, heaviest first
  int* item_q0;          // [n_items]
  int* item_tmp;         // [2 * n_items] scratch of rowmap_kernel (the unsorted list)
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool valid) {
  const int sz = valid ? 16 : 0;  // src-size 0 => 16 bytes of zeros
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_u32(smem)), "l"(gmem), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_f16_16816(float* c, const uint32_t* a, uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// byte offset of 16-byte chunk `chunk` of row `row` in a [rows][HD] 16-bit tile with XOR swizzle
template <int HD>
__device__ __forceinline__ uint32_t sw_off(int row, int chunk) {
  return static_cast<uint32_t>(row * (HD * 2) + ((chunk ^ (row & 7)) << 4));
}

// A segment of ONE row (every decode row of the paper's schedule) is not MMA-shaped: on the m16n8k16 path it fills 1 of 16
// accumulator rows and one of the CTA's four warps walks its 8-9 KV tiles alone (the legacy HMMA pipe issues one m16n8k16
// per ~13 cycles per scheduler, so these rows cost 40 % of the kernel's tensor time for 0.1 % of its FLOPs).  Such a
// (segment, head) unit keeps the kernel's cp.async K/V tile pipeline but computes each tile on plain FMAs with all 128
// threads: QK with 4 threads per position (HD / 4 dims each, q in registers) and a 2-step shuffle, the 32 scores of the
// tile through shared memory, then an online-softmax update in which thread t owns output columns [t * HD / 128, ..).
// Tiles are walked in LOGICAL position order (result independent of base_r), every reduction order is fixed.
// WIN (f3): rows see only the last `window` positions, max(0, p - window + 1)..p; positions may exceed C, slot
// (base + j) mod C then holds the newest position congruent to j (af.h: af_ring_set_window).  WIN = false is the v1 kernel.
template <int HD, bool WIN = false>
__global__ void __launch_bounds__(ATT_THREADS, 3)
attention_kernel(const act_t* __restrict__ q,     // [T, H*HD] rotated queries
                 const act_t* __restrict__ kv,    // ring, layer base: [2][R][H][C][HD]
                 act_t* __restrict__ out,         // [T, H*HD]
                 StepTables tb, int H, int R, int C, float scale_log2, int window = 0) {
  constexpr int CH = HD / 8;                  // 16-byte chunks per row
  constexpr int TILE_BYTES = ATT_BKV * HD * 2;
  extern __shared__ __align__(128) uint8_t att_smem[];
  uint8_t* sQ = att_smem;
  uint8_t* sK = sQ + ATT_BQ * HD * 2;               // ATT_STAGES stages
  uint8_t* sV = sK + ATT_STAGES * TILE_BYTES;       // ATT_STAGES stages

  pdl_wait();
  pdl_launch_dependents();
  const int item = blockIdx.y, h = blockIdx.x;  // items are sorted heaviest first; all heads of an item are neighbours
  const int seg = tb.item_seg[item], q0 = tb.item_q0[item];
  const int req = tb.seg_req[seg], start = tb.seg_start[seg], len = tb.seg_len[seg];
  const int row0 = tb.seg_row0[seg], base = tb.seg_base[seg];
  const int nq = min(ATT_BQ, len - q0);
  const int kv_end = start + q0 + nq;         // positions [0, kv_end) are visible to the tile's last row
  const int n_tiles = (kv_end + ATT_BKV - 1) / ATT_BKV;
  const int kv_lo = WIN ? max(0, start + q0 - window + 1) : 0;   // lowest position visible to the tile's first row
  const int tile_lo = WIN ? kv_lo / ATT_BKV : 0;
  const int W = WIN ? window : (1 << 30);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3;

  const size_t head_stride = static_cast<size_t>(C) * HD;
  const act_t* kbase = kv + (static_cast<size_t>(0 * R + req) * H + h) * head_stride;
  const act_t* vbase = kv + (static_cast<size_t>(1 * R + req) * H + h) * head_stride;

  const bool fma_row = !WIN && len == 1;   // a one-row segment: the FMA tile path below (block-uniform)
  __shared__ float s_scores[ATT_BKV];

  // ---- async loads: Q tile, then KV tile 0 ----
  for (int i = tid; i < ATT_BQ * CH; i += ATT_THREADS) {
    const int r = i / CH, c = i % CH;
    const bool ok = r < nq;
    const act_t* src = q + static_cast<size_t>(row0 + q0 + (ok ? r : 0)) * (H * HD) + h * HD + c * 8;
    cp_async16(sQ + sw_off<HD>(r, c), src, ok);
  }
  auto load_kv = [&](int tile, int stage) {
    const int j0 = tile * ATT_BKV;
    for (int i = tid; i < ATT_BKV * CH; i += ATT_THREADS) {
      const int r = i / CH, c = i % CH;
      const int j = j0 + r;
      const bool ok = j < kv_end && j >= kv_lo;
      int slot = base + (ok ? j : 0);
      if (WIN) slot %= C;                   // positions may exceed C
      else slot = slot >= C ? slot - C : slot;   // (base + j) mod C, base < C and j < C
      const size_t off = static_cast<size_t>(slot) * HD + c * 8;
      cp_async16(sK + stage * TILE_BYTES + sw_off<HD>(r, c), kbase + off, ok);
      cp_async16(sV + stage * TILE_BYTES + sw_off<HD>(r, c), vbase + off, ok);
    }
  };
#pragma unroll
  for (int t = 0; t < ATT_STAGES - 1; ++t) {   // prologue: the first ATT_STAGES - 1 tiles (a group each, empty past the end)
    if (tile_lo + t < n_tiles) load_kv(tile_lo + t, t);
    cp_async_commit();
  }

  float o_acc[HD / 8][4];
#pragma unroll
  for (int i = 0; i < HD / 8; ++i) { o_acc[i][0] = o_acc[i][1] = o_acc[i][2] = o_acc[i][3] = 0.f; }
  float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
  uint32_t qf[HD / 16][4];

  // warp -> (16-row strip, KV part): the two warps of a strip take alternate KV tiles and their partial (max, sum, O) are
  // merged at the end in part order - a strip's serial chain is half as long as with one warp per strip
  const int strip = warp & 1, part = warp >> 1;
  const bool warp_active = strip * 16 < nq;
  const int p_lo = start + q0 + strip * 16 + g;   // position of this thread's first row (second = +8)
  const int warp_pmin = start + q0 + strip * 16, warp_pmax = warp_pmin + 15;

  for (int tile = tile_lo; tile < n_tiles; ++tile) {
    const int stage = (tile - tile_lo) % ATT_STAGES;
    // the stage of tile + STAGES - 1 was released at the end of tile - 1
    if (tile + ATT_STAGES - 1 < n_tiles) load_kv(tile + ATT_STAGES - 1, (tile - tile_lo + ATT_STAGES - 1) % ATT_STAGES);
    cp_async_commit();
    cp_async_wait<ATT_STAGES - 1>();
    __syncthreads();
    if (tile == tile_lo) {
#pragma unroll
      for (int kk = 0; kk < HD / 16; ++kk) {
        const int r = strip * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        const int c = kk * 2 + (lane >> 4);
        ldsm_x4(smem_u32(sQ + sw_off<HD>(r, c)), qf[kk][0], qf[kk][1], qf[kk][2], qf[kk][3]);
      }
    }
    const int j0 = tile * ATT_BKV;
    if (fma_row) {
      // ---- one query row on FMAs: thread (jj = tid / 4, part = tid % 4) scores position j0 + jj over HD / 4 dims ----
      const uint8_t* cK = sK + stage * TILE_BYTES;
      const uint8_t* cV = sV + stage * TILE_BYTES;
      constexpr int CPT = CH / 4;                       // 16-byte chunks of a K row per thread
      const int jj = tid >> 2, prt = tid & 3;
      if (tile == tile_lo) {                            // q (row 0 of the Q tile) -> registers, this thread's HD / 4 dims
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
          const uint4 v = *reinterpret_cast<const uint4*>(sQ + sw_off<HD>(0, prt * CPT + c));
          qf[c][0] = v.x; qf[c][1] = v.y; qf[c][2] = v.z; qf[c][3] = v.w;
        }
      }
      float sdot = 0.f;
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const uint4 kk = *reinterpret_cast<const uint4*>(cK + sw_off<HD>(jj, prt * CPT + c));
        const uint32_t b4[4] = {kk.x, kk.y, kk.z, kk.w};
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&qf[c][m]));
          const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&b4[m]));
          sdot = fmaf(a.x, b.x, sdot); sdot = fmaf(a.y, b.y, sdot);
        }
      }
      sdot += __shfl_xor_sync(0xffffffffu, sdot, 1);
      sdot += __shfl_xor_sync(0xffffffffu, sdot, 2);
      if (prt == 0) s_scores[jj] = (j0 + jj < kv_end) ? sdot * scale_log2 : -INFINITY;
      __syncthreads();
      // online softmax: every thread scans the tile's 32 scores (broadcast reads) and updates its own output column(s)
      float mt = -INFINITY;
#pragma unroll
      for (int j = 0; j < ATT_BKV; ++j) mt = fmaxf(mt, s_scores[j]);
      const float m_new = fmaxf(m_run[0], mt);          // finite: position j0 <= own position is always visible
      const float alpha = exp2f(m_run[0] - m_new);
      m_run[0] = m_new;
      float rs = 0.f, a0 = o_acc[0][0] * alpha, a1 = o_acc[0][1] * alpha;
      const int col = (2 * tid) % HD;                   // this thread's two output columns (HD = 64: the upper half of the CTA repeats them)
#pragma unroll
      for (int j = 0; j < ATT_BKV; ++j) {
        const float pj = exp2f(s_scores[j] - m_new);
        rs += pj;
        const float2 vv = __half22float2(*reinterpret_cast<const __half2*>(cV + sw_off<HD>(j, col >> 3) + (col & 7) * 2));
        a0 = fmaf(pj, vv.x, a0); a1 = fmaf(pj, vv.y, a1);
      }
      l_run[0] = l_run[0] * alpha + rs;
      o_acc[0][0] = a0; o_acc[0][1] = a1;
    } else
    if (warp_active && ((tile - tile_lo) & 1) == part && j0 <= warp_pmax && (!WIN || j0 + ATT_BKV - 1 > warp_pmin - W)) {
      const uint8_t* cK = sK + stage * TILE_BYTES;
      const uint8_t* cV = sV + stage * TILE_BYTES;
      float s[ATT_BKV / 8][4];
#pragma unroll
      for (int i = 0; i < ATT_BKV / 8; ++i) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; }
#pragma unroll
      for (int kk = 0; kk < HD / 16; ++kk) {
#pragma unroll
        for (int nb = 0; nb < ATT_BKV / 8; nb += 2) {
          uint32_t b0, b1, b2, b3;
          const int r = nb * 8 + (lane & 7) + (lane >> 4) * 8;
          const int c = kk * 2 + ((lane >> 3) & 1);
          ldsm_x4(smem_u32(cK + sw_off<HD>(r, c)), b0, b1, b2, b3);
          mma_f16_16816(s[nb], qf[kk], b0, b1);
          mma_f16_16816(s[nb + 1], qf[kk], b2, b3);
        }
      }
      // ---- causal mask within the request + online softmax (base-2 exponent) ----
      float mx[2] = {-INFINITY, -INFINITY};
      if (j0 + ATT_BKV - 1 > warp_pmin || (WIN && j0 <= warp_pmax - W)) {   // the tile crosses the diagonal (or the window's lower edge) of one of the warp's rows
#pragma unroll
        for (int nb = 0; nb < ATT_BKV / 8; ++nb) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int j = j0 + nb * 8 + 2 * t + (e & 1);
            const int p = p_lo + (e >> 1) * 8;
            const float v = (j <= p && (!WIN || j > p - W)) ? s[nb][e] * scale_log2 : -INFINITY;
            s[nb][e] = v;
            mx[e >> 1] = fmaxf(mx[e >> 1], v);
          }
        }
      } else {                              // every position of the tile is visible to every row of the warp
#pragma unroll
        for (int nb = 0; nb < ATT_BKV / 8; ++nb) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float v = s[nb][e] * scale_log2;
            s[nb][e] = v;
            mx[e >> 1] = fmaxf(mx[e >> 1], v);
          }
        }
      }
      float alpha[2];
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        mx[r] = fmaxf(mx[r], __shfl_xor_sync(0xffffffffu, mx[r], 1));
        mx[r] = fmaxf(mx[r], __shfl_xor_sync(0xffffffffu, mx[r], 2));
        const float m_new = fmaxf(m_run[r], mx[r]);
        alpha[r] = (m_new == -INFINITY) ? 1.f : exp2f(m_run[r] - m_new);
        m_run[r] = m_new;
        mx[r] = (m_new == -INFINITY) ? 0.f : m_new;  // rows with nothing visible yet
      }
      float rs[2] = {0.f, 0.f};
#pragma unroll
      for (int nb = 0; nb < ATT_BKV / 8; ++nb) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float pv = exp2f(s[nb][e] - mx[e >> 1]);
          s[nb][e] = pv;
          rs[e >> 1] += pv;
        }
      }
#pragma unroll
      for (int r = 0; r < 2; ++r) l_run[r] = l_run[r] * alpha[r] + rs[r];
      if (__any_sync(0xffffffffu, alpha[0] != 1.f || alpha[1] != 1.f)) {   // some row's running maximum moved
#pragma unroll
        for (int i = 0; i < HD / 8; ++i) {
          o_acc[i][0] *= alpha[0]; o_acc[i][1] *= alpha[0];
          o_acc[i][2] *= alpha[1]; o_acc[i][3] *= alpha[1];
        }
      }
      // ---- O += P V ----
#pragma unroll
      for (int kk = 0; kk < ATT_BKV / 16; ++kk) {
        uint32_t a[4];
        a[0] = pack_act(s[2 * kk][0], s[2 * kk][1]);
        a[1] = pack_act(s[2 * kk][2], s[2 * kk][3]);
        a[2] = pack_act(s[2 * kk + 1][0], s[2 * kk + 1][1]);
        a[3] = pack_act(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
        for (int db = 0; db < HD / 8; db += 2) {
          uint32_t b0, b1, b2, b3;
          const int r = kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
          const int c = db + (lane >> 4);
          ldsm_x4_trans(smem_u32(cV + sw_off<HD>(r, c)), b0, b1, b2, b3);
          mma_f16_16816(o_acc[db], a, b0, b1);
          mma_f16_16816(o_acc[db + 1], a, b2, b3);
        }
      }
    }
    __syncthreads();  // everyone is done with this stage before it is refilled
  }
  cp_async_wait<0>();

  if (fma_row) {
    if (2 * tid < HD) {
      const float inv = 1.f / l_run[0];
      *reinterpret_cast<uint32_t*>(out + static_cast<size_t>(row0) * (H * HD) + h * HD + 2 * tid) = pack_act(o_acc[0][0] * inv, o_acc[0][1] * inv);
    }
    return;
  }
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    l_run[r] += __shfl_xor_sync(0xffffffffu, l_run[r], 1);
    l_run[r] += __shfl_xor_sync(0xffffffffu, l_run[r], 2);
  }
  // ---- merge the two KV parts of every strip through the (now idle) K/V stages: part 1 publishes, part 0 combines ----
  float* mo = reinterpret_cast<float*>(sK) + static_cast<size_t>(strip) * (16 * HD + 32);   // O [16][HD], then m[16], l[16]
  if (part == 1 && warp_active) {
#pragma unroll
    for (int db = 0; db < HD / 8; ++db) {
      *reinterpret_cast<float2*>(mo + g * HD + db * 8 + 2 * t) = make_float2(o_acc[db][0], o_acc[db][1]);
      *reinterpret_cast<float2*>(mo + (g + 8) * HD + db * 8 + 2 * t) = make_float2(o_acc[db][2], o_acc[db][3]);
    }
    if (t == 0) {
      mo[16 * HD + g] = m_run[0]; mo[16 * HD + g + 8] = m_run[1];
      mo[16 * HD + 16 + g] = l_run[0]; mo[16 * HD + 24 + g] = l_run[1];
    }
  }
  __syncthreads();
  if (part == 0 && warp_active) {
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const float m_o = mo[16 * HD + g + 8 * r], l_o = mo[16 * HD + 16 + g + 8 * r];
      const float m_new = fmaxf(m_run[r], m_o);
      const float a_s = (m_new == -INFINITY) ? 1.f : exp2f(m_run[r] - m_new);
      const float a_o = (m_new == -INFINITY) ? 0.f : exp2f(m_o - m_new);
      l_run[r] = l_run[r] * a_s + l_o * a_o;
      const int qi = strip * 16 + g + r * 8;
      const float inv = 1.f / l_run[r];
      act_t* dst = out + static_cast<size_t>(row0 + q0 + (qi < nq ? qi : 0)) * (H * HD) + h * HD;
#pragma unroll
      for (int db = 0; db < HD / 8; ++db) {
        const float2 ov = *reinterpret_cast<const float2*>(mo + (g + 8 * r) * HD + db * 8 + 2 * t);
        const float x0 = (o_acc[db][2 * r] * a_s + ov.x * a_o) * inv, x1 = (o_acc[db][2 * r + 1] * a_s + ov.y * a_o) * inv;
        if (qi < nq) *reinterpret_cast<uint32_t*>(dst + db * 8 + 2 * t) = pack_act(x0, x1);
      }
    }
  }
}

}  // namespace af
