// Packed-projection GEMM for sm_100a: out[token, feature] (op)= sum_k X[token, k] * W[feature, k]
// (steps a2/a5/a7/a8/a10 of SURVEY.md 8(a); Alg. 2 lines 2 and 6).
//
// "Swap-AB" orientation: the WEIGHT tile (128 output features x 64 k) is the UMMA A operand and
// the packed TOKEN tile (all T <= 288 tokens x 64 k) is the B operand, so the 282-row packed matrix of the paper's
// schedule maps onto UMMA N = 2 x 144 with 2% padding instead of 3 x 128-row M tiles with 27% padding, and a
// decode-only step (T <= 16) uses N = 16.  Both operands are K-major in global memory, are staged by TMA with the
// 128-byte swizzle, and are consumed by tcgen05.mma (kind::f16, bf16 in, fp32 accumulate in TMEM).
//
// Stream-K: the (tile, k-block) units are split evenly and contiguously over a persistent grid (<= 1 CTA per SM).
// A CTA that holds the k-tail of a tile writes its fp32 partial to the workspace and raises a flag; the CTA that
// holds the k-head (processed LAST in its own range, so the partials are already there) adds the partials in CTA
// order (deterministic) and runs the epilogue.
//
// Warp roles (192 threads): warps 0-3 epilogue (TMEM lane quadrant = warp id), warp 4 TMA producer, warp 5 MMA issuer.
#pragma once
#include "ptx.cuh"

namespace af {

constexpr int GEMM_BM = 128;       // weight rows (output features) per tile = UMMA M
constexpr int GEMM_BK = 64;        // bf16 elements per k-block = one 128-byte swizzle row
constexpr int GEMM_THREADS = 192;
constexpr int GEMM_MAX_TOK = 288;  // tokens per launch (two UMMA N halves of <= 144, or one of <= 256)
constexpr int GEMM_TMEM_COLS = 512;

enum GemmEpilogue : int { EPI_STORE_BF16 = 0, EPI_RESIDUAL_F32 = 1, EPI_STORE_F32 = 2 };

struct GemmParams {
  int n_parts;         // weight matrices stacked along the feature axis (q|k|v, gate|up): 1..3
  int part_rows;       // output features per part
  int tiles_per_part;  // ceil(part_rows / 128)
  int K;               // reduction length
  int num_kb;          // ceil(K / 64)
  int T;               // valid tokens of this launch
  int tok0;            // first token row (row coordinate into X and out)
  int n1, n2;          // UMMA N of the two token halves (multiples of 16, n2 may be 0)
  int total_units;     // n_parts * tiles_per_part * num_kb
  int units_per_cta;
  int stages;
  int epi;             // GemmEpilogue
  void* out;           // [tokens, ld_out] bf16 or fp32
  int ld_out;
  float* partial;      // [grid][n1+n2][128] fp32 stream-K partials
  int* flags;          // [grid] epoch flags
  int epoch;
};

__device__ __forceinline__ void gemm_epilogue_store(const GemmParams& p, int epi, int feat, bool feat_ok, int c0,
                                                    const float* v) {
  if (!feat_ok) return;
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const int c = c0 + j;
    if (c < p.T) {
      const size_t o = static_cast<size_t>(p.tok0 + c) * p.ld_out + feat;
      if (epi == EPI_STORE_BF16) {
        reinterpret_cast<__nv_bfloat16*>(p.out)[o] = __float2bfloat16_rn(v[j]);
      } else if (epi == EPI_RESIDUAL_F32) {
        float* dst = reinterpret_cast<float*>(p.out) + o;
        *dst = *dst + v[j];
      } else {
        reinterpret_cast<float*>(p.out)[o] = v[j];
      }
    }
  }
}

__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ CUtensorMap map_w0, const __grid_constant__ CUtensorMap map_w1,
                    const __grid_constant__ CUtensorMap map_w2, const __grid_constant__ CUtensorMap map_x,
                    const GemmParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte aligned tile area (the 128-byte swizzle pattern repeats every 1024 bytes)
  uint8_t* tiles = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int n_pad = p.n1 + p.n2;
  const uint32_t a_bytes = GEMM_BM * GEMM_BK * 2;
  const uint32_t b_bytes = static_cast<uint32_t>(n_pad) * GEMM_BK * 2;
  const uint32_t stage_bytes = a_bytes + b_bytes;

  __shared__ uint64_t full_bar[12], empty_bar[12], tmem_full_bar, tmem_empty_bar;
  __shared__ uint32_t tmem_base_smem;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int cta = blockIdx.x;

  if (warp == 4 && lane == 0) {
    tma_prefetch_desc(&map_w0);
    if (p.n_parts > 1) tma_prefetch_desc(&map_w1);
    if (p.n_parts > 2) tma_prefetch_desc(&map_w2);
    tma_prefetch_desc(&map_x);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
    }
    mbar_init(&tmem_full_bar, 1);
    mbar_init(&tmem_empty_bar, 4);
    fence_barrier_init();
  }
  if (warp == 5) tmem_alloc(&tmem_base_smem, GEMM_TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  const int u_begin = min(cta * p.units_per_cta, p.total_units);
  const int u_end = min(u_begin + p.units_per_cta, p.total_units);

  pdl_wait();  // everything above overlaps the previous kernel's tail when launched with PDL

  if (warp == 4) {
    // ================================ TMA producer ================================
    if (lane == 0) {
      const uint64_t pol_w = policy_evict_first();  // weights are streamed once per step
      const uint64_t pol_x = policy_evict_last();   // the packed activations are re-read by every CTA
      int stage = 0;
      uint32_t phase = 0;
      for (int u = u_begin; u < u_end; ++u) {
        const int tile = u / p.num_kb, kb = u - tile * p.num_kb;
        const int part = tile / p.tiles_per_part, tip = tile - part * p.tiles_per_part;
        const CUtensorMap* mw = part == 0 ? &map_w0 : (part == 1 ? &map_w1 : &map_w2);
        mbar_wait(&empty_bar[stage], phase ^ 1);
        uint8_t* sa = tiles + static_cast<size_t>(stage) * stage_bytes;
        uint8_t* sb = sa + a_bytes;
        mbar_arrive_expect_tx(&full_bar[stage], stage_bytes);
        tma_load_2d(sa, mw, &full_bar[stage], kb * GEMM_BK, tip * GEMM_BM, pol_w);
        tma_load_2d(sb, &map_x, &full_bar[stage], kb * GEMM_BK, p.tok0, pol_x);
        if (p.n2 > 0)
          tma_load_2d(sb + static_cast<size_t>(p.n1) * GEMM_BK * 2, &map_x, &full_bar[stage], kb * GEMM_BK,
                      p.tok0 + p.n1, pol_x);
        if (++stage == p.stages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 5) {
    // ================================ MMA issuer (one thread) ================================
    if (lane == 0) {
      const uint32_t idesc1 = umma_idesc_bf16(GEMM_BM, p.n1);
      const uint32_t idesc2 = umma_idesc_bf16(GEMM_BM, p.n2 > 0 ? p.n2 : 16);
      int stage = 0;
      uint32_t phase = 0, acc_phase = 0;
      int u = u_begin;
      while (u < u_end) {
        const int tile = u / p.num_kb, kb0 = u - tile * p.num_kb;
        const int kb1 = min(p.num_kb, kb0 + (u_end - u));
        mbar_wait(&tmem_empty_bar, acc_phase ^ 1);  // epilogue has drained the accumulator
        tc_fence_after();
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(tiles + static_cast<size_t>(stage) * stage_bytes);
          const uint32_t sb = sa + a_bytes;
          const uint64_t da = umma_smem_desc_sw128(sa);
          const uint64_t db1 = umma_smem_desc_sw128(sb);
          const uint64_t db2 = umma_smem_desc_sw128(sb + p.n1 * GEMM_BK * 2);
#pragma unroll
          for (int k = 0; k < GEMM_BK / 16; ++k) {
            const uint32_t accum = (kb > kb0 || k > 0) ? 1u : 0u;
            // advancing 16 bf16 = 32 bytes along K inside the swizzle row: +2 in the (addr >> 4) field
            umma_bf16(tmem_base, da + 2 * k, db1 + 2 * k, idesc1, accum);
            if (p.n2 > 0) umma_bf16(tmem_base + p.n1, da + 2 * k, db2 + 2 * k, idesc2, accum);
          }
          umma_commit(&empty_bar[stage]);  // frees the smem slot when these MMAs have read it
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
        umma_commit(&tmem_full_bar);  // accumulator complete -> epilogue
        acc_phase ^= 1;
        u += kb1 - kb0;
      }
    }
  } else {
    // ================================ epilogue warps 0..3 ================================
    const int quad = warp;  // TMEM lanes [32*quad, 32*quad+32)
    const int row = quad * 32 + lane;
    uint32_t acc_phase = 0;
    int u = u_begin;
    while (u < u_end) {
      const int tile = u / p.num_kb, kb0 = u - tile * p.num_kb;
      const int kb1 = min(p.num_kb, kb0 + (u_end - u));
      const int part = tile / p.tiles_per_part, tip = tile - part * p.tiles_per_part;
      const int feat_in_part = tip * GEMM_BM + row;
      const bool feat_ok = feat_in_part < p.part_rows;
      const int feat = part * p.part_rows + feat_in_part;
      const bool contributor = kb0 > 0;
      const bool owner_partial = (kb0 == 0) && (kb1 < p.num_kb);
      int c_first = 0, c_last = -1;
      if (owner_partial) {
        // CTAs holding the rest of this tile: cta+1 .. while their range starts before the tile ends
        c_first = cta + 1;
        const int tile_end = (tile + 1) * p.num_kb;
        c_last = min((tile_end - 1) / p.units_per_cta, static_cast<int>(gridDim.x) - 1);
        if (lane == 0) {
          for (int c = c_first; c <= c_last; ++c) {
            while (*reinterpret_cast<volatile int*>(p.flags + c) != p.epoch) {
            }
          }
          __threadfence();
        }
        __syncwarp();
      }
      mbar_wait(&tmem_full_bar, acc_phase);
      tc_fence_after();
      float* my_partial = p.partial + static_cast<size_t>(cta) * n_pad * GEMM_BM;
      for (int c0 = 0; c0 < n_pad && c0 < p.T; c0 += 16) {
        uint32_t r[16];
        tmem_ld16(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + c0, r);
        tmem_ld_wait();
        float v[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = __uint_as_float(r[j]);
        if (contributor) {
#pragma unroll
          for (int j = 0; j < 16; ++j) my_partial[static_cast<size_t>(c0 + j) * GEMM_BM + row] = v[j];
        } else {
          for (int c = c_first; c <= c_last; ++c) {
            const float* q = p.partial + static_cast<size_t>(c) * n_pad * GEMM_BM;
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] += __ldcg(q + static_cast<size_t>(c0 + j) * GEMM_BM + row);
          }
          gemm_epilogue_store(p, p.epi, feat, feat_ok, c0, v);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tmem_empty_bar);
      if (contributor) {
        __threadfence();
        asm volatile("bar.sync 1, 128;\n" ::: "memory");  // the 4 epilogue warps only
        if (threadIdx.x == 0) {
          __threadfence();
          atomicExch(p.flags + cta, p.epoch);
        }
      }
      acc_phase ^= 1;
      u += kb1 - kb0;
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 5) {
    tc_fence_after();
    tmem_dealloc(tmem_base, GEMM_TMEM_COLS);
  }
}

}  // namespace af
