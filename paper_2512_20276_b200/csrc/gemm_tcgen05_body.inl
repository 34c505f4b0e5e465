// Body of gemm_tcgen05.cuh (kept in a second file only to keep each file short); see the header for the design.

template <bool kMma2, bool kFrag>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ CUtensorMap map_w0, const __grid_constant__ CUtensorMap map_w1,
                    const __grid_constant__ CUtensorMap map_w2, const __grid_constant__ CUtensorMap map_x,
                    const __grid_constant__ CUtensorMap map_out, const __grid_constant__ CUtensorMap map_part,
                    const GemmParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte aligned tile area (the 128-byte swizzle pattern repeats every 1024 bytes)
  // (offset arithmetic on the __shared__ array, not an integer round trip, so the compiler keeps the shared address space)
  uint8_t* tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int n_pad = p.n1 + p.n2;
  const uint32_t a_bytes = GEMM_BM * GEMM_BK * 2;
  // mma2: one tcgen05.mma.cta_group::2 per CTA pair (M = 256 = the two CTAs' weight tiles); each CTA stages only HALF
  // of the activation rows of every UMMA-N half, so a stage is 34 KB instead of 52 KB at T = 282
  constexpr bool mma2 = kMma2;  // (a second instantiation: a kernel holding cta_group::2 instructions must be launched in clusters)
  const uint32_t b_bytes = static_cast<uint32_t>(mma2 ? n_pad / 2 : n_pad) * GEMM_BK * 2;
  const uint32_t stage_bytes = a_bytes + b_bytes;
  float* xch = reinterpret_cast<float*>(tiles + static_cast<size_t>(p.stages) * stage_bytes);

  __shared__ uint64_t full_bar[GEMM_MAX_STAGES], conv_bar[GEMM_MAX_STAGES], empty_bar[GEMM_MAX_STAGES], tmem_full_bar,
      tmem_empty_bar, fix_bar;
  __shared__ uint32_t tmem_base_smem;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int cta = blockIdx.x;
  // 2-CTA cluster: both CTAs sweep the same k-blocks of two neighbouring weight tiles and each loads one half of the
  // activation k-block, multicast into both (halves the L2 -> SM traffic of the operand every CTA needs in full)
  const int crank = p.cluster > 1 ? static_cast<int>(cluster_ctarank()) : 0;
  // Work is split over clusters (unit = (tile pair, k-block)).  Schedule row n_cl - 1 - (launch order): a stream-K
  // owner waits for contributor pieces of HIGHER schedule rows, i.e. of clusters that were dispatched EARLIER, so a
  // waiting CTA never depends on one that is not yet resident (no deadlock when the grid is only partly resident).
  const int cl = p.n_cl - 1 - cta / p.cluster;

  // the first use of this cluster's piece list (a dependent global load in front of the first TMA request) would cost
  // ~0.8 us after the cluster barrier: pull its line into L1 now
  if (lane == 0) asm volatile("prefetch.global.L1 [%0];\n" ::"l"(p.sched + static_cast<size_t>(cl) * GEMM_MAX_PIECES));
  if (warp == GEMM_EPI_WARPS && lane == 0) {
    tma_prefetch_desc(&map_w0);
    if (p.n_parts > 1 || p.a_pair == 1) tma_prefetch_desc(&map_w1);
    if (p.n_parts > 2) tma_prefetch_desc(&map_w2);
    tma_prefetch_desc(&map_x);
    tma_prefetch_desc(&map_out);
    tma_prefetch_desc(&map_part);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&conv_bar[s], GEMM_EPI_WARPS);
      mbar_init(&empty_bar[s], mma2 ? 1 : p.cluster);
    }
    mbar_init(&tmem_full_bar, 1);
    mbar_init(&tmem_empty_bar, mma2 ? 2 * GEMM_EPI_WARPS : GEMM_EPI_WARPS);  // mma2: the leader waits for both drains
    mbar_init(&fix_bar, 1);
    fence_barrier_init();
  }
  if (warp == GEMM_EPI_WARPS + 1) {
    if (mma2) tmem_alloc_cg2(&tmem_base_smem, GEMM_TMEM_COLS); else tmem_alloc(&tmem_base_smem, GEMM_TMEM_COLS);
  }
  tc_fence_before();
  __syncthreads();
  if (p.cluster > 1) cluster_sync();  // the peer's barriers exist before anything is multicast to them
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  pdl_launch_dependents();  // dependents still wait (griddepcontrol.wait) for this whole grid before reading its output

  // this cluster's pieces (host-built schedule, see GemmPiece): every role walks the same list
  const GemmPiece* my_pieces = p.sched + static_cast<size_t>(cl) * GEMM_MAX_PIECES;
  auto get_piece = [&](int i) {
    GemmPiece pc;
    const int4* src = reinterpret_cast<const int4*>(my_pieces + i);
    *reinterpret_cast<int4*>(&pc) = __ldg(src);
    *(reinterpret_cast<int4*>(&pc) + 1) = __ldg(src + 1);
    return pc;
  };

  if (warp == GEMM_EPI_WARPS) {
    // ================================ TMA producer ================================
    if (lane == 0) {
      const uint64_t pol_w = policy_evict_first();  // weights are streamed once per step
      const uint64_t pol_x = policy_evict_last();   // the packed activations are re-read by every CTA
      // (pair, kb) of the unit being loaded, advanced incrementally: no division in the steady-state loop
      int l_pi = -1, l_pair = 0, l_kb = 0, l_kb1 = 0;   // cursor over the (piece, k-block) units that need loads
      bool l_more = true;
      const CUtensorMap* l_mw = &map_w0;
      int l_row = 0;   // first weight row of this CTA's tile in its matrix
      auto set_tile = [&]() {
        const int tile = min(l_pair * p.cluster + crank, p.n_tiles - 1);  // (an odd tile count: reload the last)
        if (p.a_pair) {
          l_row = tile * (p.a_pair == 2 ? GEMM_BM : 64);   // (2: gate | up interleaved at load time, 128 rows per tile)
        } else {
          const int part = tile / p.tiles_per_part;
          l_mw = part == 0 ? &map_w0 : (part == 1 ? &map_w1 : &map_w2);
          l_row = (tile - part * p.tiles_per_part) * GEMM_BM;
        }
      };
      auto next_piece = [&]() {   // move the cursor to the next piece that has k-blocks
        while (true) {
          if (++l_pi >= GEMM_MAX_PIECES) { l_more = false; return; }
          const GemmPiece pc = get_piece(l_pi);
          if (pc.pair < 0) { l_more = false; return; }
          if (pc.kb1 > pc.kb0) { l_pair = pc.pair; l_kb = pc.kb0; l_kb1 = pc.kb1; set_tile(); return; }
        }
      };
      next_piece();
      auto advance = [&]() {
        if (++l_kb == l_kb1) next_piece();
      };
      auto load_w = [&](int stage) {
        uint8_t* sa = tiles + static_cast<size_t>(stage) * stage_bytes;
        const int kc = l_kb * GEMM_BK;
        if (p.a_pair == 1) {  // every TMEM lane quadrant = 16 gate rows + the 16 up rows of the same features
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            if (mma2) {
              tma_load_2d_cg2(sa + q * 4096, &map_w0, &full_bar[stage], kc, l_row + q * 16, pol_w);
              tma_load_2d_cg2(sa + q * 4096 + 2048, &map_w1, &full_bar[stage], kc, l_row + q * 16, pol_w);
            } else {
              tma_load_2d(sa + q * 4096, &map_w0, &full_bar[stage], kc, l_row + q * 16, pol_w);
              tma_load_2d(sa + q * 4096 + 2048, &map_w1, &full_bar[stage], kc, l_row + q * 16, pol_w);
            }
          }
        } else {
          if (mma2) tma_load_2d_cg2(sa, l_mw, &full_bar[stage], kc, l_row, pol_w);
          else tma_load_2d(sa, l_mw, &full_bar[stage], kc, l_row, pol_w);
        }
      };
      // the activation k-block = two boxes of p.xh token rows; in a cluster CTA r loads box r for both CTAs
      auto load_x = [&](int kb, int stage) {
        uint8_t* sb = tiles + static_cast<size_t>(stage) * stage_bytes + a_bytes;
        const size_t half = static_cast<size_t>(p.xh) * GEMM_BK * 2;
        if (mma2) {  // this CTA's half of the rows of each UMMA-N half (the map's box is n1 / 2 rows)
          const int h1 = p.n1 / 2;
          tma_load_2d_cg2(sb, &map_x, &full_bar[stage], kb * GEMM_BK, p.tok0 + crank * h1, pol_x);
          if (p.n2 > 0)
            tma_load_2d_cg2(sb + static_cast<size_t>(h1) * GEMM_BK * 2, &map_x, &full_bar[stage], kb * GEMM_BK,
                            p.tok0 + p.n1 + crank * h1, pol_x);
        } else if (p.cluster > 1) {
          tma_load_2d_mc(sb + crank * half, &map_x, &full_bar[stage], kb * GEMM_BK, p.tok0 + crank * p.xh, 0x3, pol_x);
        } else {
          tma_load_2d(sb, &map_x, &full_bar[stage], kb * GEMM_BK, p.tok0, pol_x);
          tma_load_2d(sb + half, &map_x, &full_bar[stage], kb * GEMM_BK, p.tok0 + p.xh, pol_x);
        }
      };
      // The weights do not depend on the previous kernel: start streaming the first p.w_pre stages before the PDL
      // dependency resolves (not all of them: the previous kernel's last CTAs still need the memory system).
      int n_pre = 0;
      int kb_pre[GEMM_MAX_STAGES];
      while (n_pre < p.w_pre && l_more) {
        if (!mma2) mbar_arrive_expect_tx(&full_bar[n_pre], stage_bytes);
        else if (crank == 0) mbar_arrive_expect_tx(&full_bar[n_pre], 2 * stage_bytes);
        load_w(n_pre);
        kb_pre[n_pre] = l_kb;
        advance();
        ++n_pre;
      }
      pdl_wait();
      for (int i = 0; i < n_pre; ++i) load_x(kb_pre[i], i);
      int stage = n_pre == p.stages ? 0 : n_pre;
      uint32_t phase = n_pre == p.stages ? 1 : 0;
      while (l_more) {
        mbar_wait(&empty_bar[stage], phase ^ 1);
        if (!mma2) mbar_arrive_expect_tx(&full_bar[stage], stage_bytes);
        else if (crank == 0) mbar_arrive_expect_tx(&full_bar[stage], 2 * stage_bytes);
        load_w(stage);
        load_x(l_kb, stage);
        advance();
        if (++stage == p.stages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == GEMM_EPI_WARPS + 1) {
    // ================================ MMA issuer (one thread) ================================
    if (lane == 0 && !(mma2 && crank != 0)) {   // mma2: only the pair's leader issues
      const uint32_t idesc1 = umma_idesc_f16(mma2 ? 2 * GEMM_BM : GEMM_BM, p.n1);
      const uint32_t idesc2 = umma_idesc_f16(mma2 ? 2 * GEMM_BM : GEMM_BM, p.n2 > 0 ? p.n2 : 16);
      int stage = 0;
      uint32_t phase = 0, acc_phase = 0;
      for (int pi = 0; pi < GEMM_MAX_PIECES; ++pi) {
        const GemmPiece pc = get_piece(pi);
        if (pc.pair < 0) break;
        const int kb0 = pc.kb0, kb1 = pc.kb1;
        if (kb1 <= kb0) continue;                   // a reduce-only piece: nothing to multiply
        mbar_wait(&tmem_empty_bar, acc_phase ^ 1);  // epilogue has drained the accumulator
        tc_fence_after();
        for (int kb = kb0; kb < kb1; ++kb) {
          // the stage has landed (and, for bf16 weights, the epilogue warps have rewritten the W tile as fp16)
          mbar_wait(p.w_fp16 ? &full_bar[stage] : &conv_bar[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(tiles + static_cast<size_t>(stage) * stage_bytes);
          const uint32_t sb = sa + a_bytes;
          const uint64_t da = umma_smem_desc_sw128(sa);
          const uint64_t db1 = umma_smem_desc_sw128(sb);
          const uint64_t db2 = umma_smem_desc_sw128(sb + (mma2 ? p.n1 / 2 : p.n1) * GEMM_BK * 2);
#pragma unroll
          for (int k = 0; k < GEMM_BK / 16; ++k) {
            const uint32_t accum = (kb > kb0 || k > 0) ? 1u : 0u;
            // advancing 16 bf16 = 32 bytes along K inside the swizzle row: +2 in the (addr >> 4) field
            if (mma2) {
              umma_f16_cg2(tmem_base, da + 2 * k, db1 + 2 * k, idesc1, accum);
              if (p.n2 > 0) umma_f16_cg2(tmem_base + p.n1, da + 2 * k, db2 + 2 * k, idesc2, accum);
            } else {
            umma_f16_cg1(tmem_base, da + 2 * k, db1 + 2 * k, idesc1, accum);
            if (p.n2 > 0) umma_f16_cg1(tmem_base + p.n1, da + 2 * k, db2 + 2 * k, idesc2, accum);
            }
          }
          // frees the smem slot when these MMAs have read it (in a cluster: in both CTAs, the peer multicasts into it)
          if (mma2) umma_commit_cg2_mc(&empty_bar[stage], 0x3);
          else if (p.cluster > 1) umma_commit_mc(&empty_bar[stage], 0x3);
          else umma_commit(&empty_bar[stage]);
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
        if (mma2) umma_commit_cg2_mc(&tmem_full_bar, 0x3); else umma_commit(&tmem_full_bar);  // accumulator -> epilogue
        acc_phase ^= 1;
      }
    }
  } else {
    // ================================ epilogue warps 0..7 ================================
    // Warp w reads TMEM lanes [32*(w%4), +32) = 32 output features; the two warps of a quadrant alternate 32-token
    // chunks.  Per chunk: TMEM -> registers -> the warp's private staging buffer -> global ([tokens][features] rows;
    // 16-byte global stores for fp16 outputs, TMA tensor stores for fp32, see gemm_tcgen05.cuh).  No epilogue warp
    // waits for another (except for the stream-K fix-up loads).
    const int quad = warp & 3, par = warp >> 2;
    const int row = quad * 32 + lane;
    const int etid = threadIdx.x;  // 0..255
    uint8_t* stg_base = reinterpret_cast<uint8_t*>(xch) + warp * (p.stg_bytes * p.stg_bufs);
    // 16-bit outputs (every GEMM of the forward) are drained in the mma fragment layout: tcgen05.ld.16x256b gives thread
    // t (feature t/4 [+8], tokens 2(t%4), +1 of every 8), which is what stmatrix.trans writes as [token][feature] rows.
    // Byte offset of this lane's row address inside a staging image (token group 0; the others are + 512 bytes):
    constexpr bool frag = kFrag;   // == (p.out_f16 != 0), a template parameter so that each variant holds one epilogue
    const uint32_t frag_off64 = (lane & 7) * 64 + (((lane >> 3) ^ ((lane & 7) >> 1)) << 4);   // 64-byte rows, SWIZZLE_64B
    const uint32_t frag_off32 = ((lane >> 4) * 8 + (lane & 7)) * 32 + ((((lane >> 3) & 1) ^ ((lane & 7) >> 2)) << 4);  // 32-byte rows, SWIZZLE_32B
    // ... and of the 16-byte piece this lane reads back and stores: token lane/4 (+ 8 per group), features 8(lane%4).. for
    // 64-byte rows; token lane/2 (+ 16 per half), features 8(lane%2).. for the 32-byte rows of the SwiGLU output
    const uint32_t rb_off64 = (lane >> 2) * 64 + (((lane & 3) ^ ((lane >> 3) & 3)) << 4);
    const uint32_t rb_off32 = (lane >> 1) * 32 + (((lane & 1) ^ ((lane >> 3) & 1)) << 4);
    uint32_t n_st = 0;  // TMA stores issued by this warp; buffer = n_st & 1
    bool store_ok = true;
#define stg (stg_base + (p.stg_bufs > 1 ? (n_st & 1) * p.stg_bytes : 0))
    auto stage_free = [&]() {  // the TMA stores issued by this warp have finished reading the staging buffer
      if (lane == 0) {  // all stores but the latest (which reads the other buffer, if there are two) are done reading
        if (p.stg_bufs > 1) bulk_wait_read<1>(); else bulk_wait_read<0>();
      }
      __syncwarp();
    };
    auto stage_store = [&](const CUtensorMap* m, int c0_, int c1_, int c2_) {
      fence_proxy_async();
      __syncwarp();
      if (lane == 0 && store_ok) {
        tma_store_3d(m, stg, c0_, c1_, c2_);
        bulk_commit();
      }
      ++n_st;
    };
    pdl_wait();
    int piece = 0;
    const int stage_area = p.stages * static_cast<int>(stage_bytes);
    uint32_t acc_phase = 0, fix_phase = 0, cphase = 0;
    int cstage = 0;
    for (int pi = 0; pi < GEMM_MAX_PIECES; ++pi) {
      const GemmPiece pc = get_piece(pi);
      if (pc.pair < 0) break;
      const int pair = pc.pair, kb0 = pc.kb0, kb1 = pc.kb1;
      const bool has_mma = kb1 > kb0;             // false: a reduce-only owner piece (its whole tile was computed by others)
      const int tile = pair * p.cluster + crank;
      const bool tile_valid = tile < p.n_tiles;   // (an odd tile count leaves the last cluster's second CTA idle)
      const bool contributor = pc.kind == PK_CONTRIB;
      const int my_slot = pc.slot * p.cluster + crank;   // contributor: where its partial and flag go
      // ---- weight transform: this piece's W stages bf16 -> fp16, in place, as they land (exact for every finite
      //      bf16 weight below 65504 in magnitude; values under 2^-14 keep 10 + e bits as fp16 subnormals) ----
      for (int kb = p.w_fp16 ? kb1 : kb0; kb < kb1; ++kb) {
        mbar_wait(&full_bar[cstage], cphase);
        uint4* wst = reinterpret_cast<uint4*>(tiles + static_cast<size_t>(cstage) * stage_bytes);
#pragma unroll
        for (int i = etid; i < static_cast<int>(a_bytes / 16); i += GEMM_EPI_WARPS * 32) {
          uint4 raw = wst[i];
          raw.x = bf16x2_to_f16x2(raw.x); raw.y = bf16x2_to_f16x2(raw.y);
          raw.z = bf16x2_to_f16x2(raw.z); raw.w = bf16x2_to_f16x2(raw.w);
          wst[i] = raw;
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive(&conv_bar[cstage]);
        if (++cstage == p.stages) { cstage = 0; cphase ^= 1; }
      }
      int c_first = 0, n_contrib = 0;
      if (pc.kind == PK_OWNER) {
        // the rest of this tile was (or is being) computed by the contributor pieces in slots [slot, slot + n_contrib)
        c_first = pc.slot; n_contrib = pc.n_contrib;
        if (etid < n_contrib) {
          volatile int* f = p.flags + (c_first + etid) * p.cluster + crank;
          SpinGuard sg;
          while (*f == 0) sg.poll();
          *f = 0;  // one consumer per flag: ready for the next launch (graph-replay safe)
          __threadfence();
        }
        AF_EPI_BAR();
      }
      store_ok = tile_valid;
      // ---- tile-uniform store coordinates: (feature, middle, token) of map_out ----
      int f0, mid;
      if (p.a_pair) {
        f0 = tile * 64 + quad * 16; mid = 0;
      } else {
        const int part = tile / p.tiles_per_part;
        f0 = (tile - part * p.tiles_per_part) * GEMM_BM + quad * 32;
        mid = p.split == SPLIT_K ? pc.mid : part;
      }
      // fp16 outputs: this lane's 16-byte piece of every row it stores (EPI_STORE: token lane/4 + 8g, features
      // 8(lane%4)..; EPI_SWIGLU: token lane/2 + 16j, features 8(lane%2)..) - pointer and guards hoisted out of the chunks
      const int st_sh = p.epi == EPI_SWIGLU ? 1 : 2;
      const int st_feat = f0 + 8 * (lane & ((1 << st_sh) - 1)), st_tok = lane >> st_sh;
      const bool st_ok = frag && store_ok && st_feat < p.out_features;
      act_t* const st_ptr = reinterpret_cast<act_t*>(p.out) + static_cast<size_t>(mid) * p.out_ld_mid + st_feat +
                            static_cast<size_t>(p.tok0 + st_tok) * p.out_ld_tok;
      // column blocks: with contributors, their partial columns [b0, b1) are bulk-copied into the (now idle) stages,
      // all contributors at once, or (a tile cut into very many pieces) `grp` at a time over 64-column blocks
      int blk_cols = n_pad, grp = n_contrib, n_groups = n_contrib > 0 ? 1 : 0;
      if (n_contrib > 0) {
        const int pe = p.part_f16 ? 2 : 4;   // bytes per partial element
        const int grp_max = stage_area / (GEMM_BLK * GEMM_BM * pe);
        if (n_contrib > grp_max) {
          grp = grp_max; blk_cols = GEMM_BLK; n_groups = (n_contrib + grp - 1) / grp;
        } else {
          blk_cols = (stage_area / (n_contrib * GEMM_BM * pe)) / GEMM_BLK * GEMM_BLK;
          if (blk_cols > n_pad) blk_cols = n_pad;
        }
      }
      const uint8_t* fix = tiles;
      bool fix_used = false;
      auto load_group = [&](int g0, int cnt, int b0, int b1) {
        if (fix_used) AF_EPI_BAR();  // everyone is done reading what the buffer held
        fix_used = true;
        if (etid == 0) {
          const uint32_t pe = p.part_f16 ? 2 : 4;
          const uint32_t bytes = static_cast<uint32_t>(frag ? ((b1 - b0 + 31) & ~31) : b1 - b0) * GEMM_BM * pe;
          fence_proxy_async_all();
          mbar_arrive_expect_tx(&fix_bar, bytes * cnt);
          for (int c = 0; c < cnt; ++c)
            bulk_load_1d(tiles + static_cast<size_t>(c) * bytes,
                         reinterpret_cast<const uint8_t*>(p.partial) +
                             (static_cast<size_t>((c_first + g0 + c) * p.cluster + crank) * GEMM_MAX_TOK + b0) * GEMM_BM * pe,
                         bytes,
                         &fix_bar);
        }
        mbar_wait(&fix_bar, fix_phase);
        fix_phase ^= 1;
      };
      auto load_acc = [&](int c0, int cw, float* v) {
        if (!has_mma) {
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = 0.f;
          return;
        }
        uint32_t r[32];
        const uint32_t ta = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + c0;
        if (frag) {   // fragment layout: r[0..15] = lanes [0, 16) of the quadrant, r[16..31] = lanes [16, 32)
          tmem_ld_frag32(ta, r);
          tmem_ld_frag32(ta + (16u << 16), r + 16);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
          return;
        }
        tmem_ld16(ta, r);
        if (cw > 16) tmem_ld16(ta + 16, r + 16);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
      };
      auto add_fix = [&](int cnt, int b0, int b1, int c0, float* v) {
        // (a 16-wide last chunk over-reads 16 columns of the staging area; those columns are never stored)
        if (frag) {   // fp16 images [chunk][quadrant][2 KB], read back in the layout they were written from
          const uint32_t img0 = smem_u32(fix) + static_cast<uint32_t>(((c0 - b0) >> 5) * 4 + quad) * 2048u + frag_off64;
          const uint32_t img_stride = static_cast<uint32_t>((b1 - b0 + 31) & ~31) * GEMM_BM * 2;
          for (int c = 0; c < cnt; ++c) {
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              uint32_t q[4];
              ldmatrix_x4_trans(img0 + c * img_stride + g * 512, q[0], q[1], q[2], q[3]);
#pragma unroll
              for (int m = 0; m < 4; ++m) {
                const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&q[m]));
                v[(m >> 1) * 16 + 4 * g + (m & 1) * 2] += f.x;
                v[(m >> 1) * 16 + 4 * g + (m & 1) * 2 + 1] += f.y;
              }
            }
          }
          return;
        }
        for (int c = 0; c < cnt; ++c) {
          const size_t e0 = (static_cast<size_t>(c) * (b1 - b0) + (c0 - b0)) * GEMM_BM + row;
#pragma unroll
          for (int h2 = 0; h2 < 2; ++h2) {
            float t[16];
            const float* q = reinterpret_cast<const float*>(fix) + e0;
#pragma unroll
            for (int j = 0; j < 16; ++j) t[j] = q[(h2 * 16 + j) * GEMM_BM];
#pragma unroll
            for (int j = 0; j < 16; ++j) v[h2 * 16 + j] += t[j];
          }
        }
      };
      auto finish_chunk = [&](int c0, int cw, float* v) {
        if (frag && (contributor || p.epi == EPI_STORE)) {
          // 32 features x 32 tokens as fp16: four stmatrix.trans write the warp's 2 KB staging image [token][feature]
          // (64-byte rows, chunk-XOR swizzle), which is read back row-wise and stored with 16-byte global stores:
          // a partial goes out as the raw image, the output as 64 contiguous bytes per token.  No TMA store, so
          // nothing to wait for before the buffer is reused but the warp's own read-back.
          __syncwarp();
          const uint32_t sa = smem_u32(stg_base);
#pragma unroll
          for (int g = 0; g < 4; ++g)
            stmatrix_x4_trans(sa + frag_off64 + g * 512, pack_act(v[4 * g], v[4 * g + 1]), pack_act(v[4 * g + 2], v[4 * g + 3]),
                              pack_act(v[16 + 4 * g], v[16 + 4 * g + 1]), pack_act(v[16 + 4 * g + 2], v[16 + 4 * g + 3]));
          __syncwarp();
          if (contributor) {
            uint8_t* dst = reinterpret_cast<uint8_t*>(p.partial) +
                           (static_cast<size_t>(my_slot) * (GEMM_MAX_TOK / 32) * 4 + (c0 >> 5) * 4 + quad) * 2048 + lane * 16;
#pragma unroll
            for (int g = 0; g < 4; ++g)
              if (store_ok) *reinterpret_cast<uint4*>(dst + g * 512) = lds128(sa + lane * 16 + g * 512);
          } else {
            act_t* dst = st_ptr + static_cast<size_t>(c0) * p.out_ld_tok;
            const int n_ok = p.T - c0 - st_tok;   // rows 8g of this lane with 8g < n_ok exist
#pragma unroll
            for (int g = 0; g < 4; ++g)
              if (st_ok && 8 * g < n_ok)
                *reinterpret_cast<uint4*>(dst + static_cast<size_t>(8 * g) * p.out_ld_tok) = lds128(sa + rb_off64 + g * 512);
          }
        } else if (frag) {
          // EPI_SWIGLU: lanes [0,16) of the quadrant hold gate, lanes [16,32) up of the same 16 features, so v[j] and
          // v[16 + j] are gate and up of one (feature, token).  16 features x 32 tokens, 32-byte rows.
          uint32_t h[8];
#pragma unroll
          for (int j = 0; j < 16; j += 2) {
            const float g0 = v[j], g1 = v[j + 1];
            const float h0 = __fdividef(g0, 1.f + __expf(-g0)) * v[16 + j], h1 = __fdividef(g1, 1.f + __expf(-g1)) * v[17 + j];
            h[j >> 1] = pack_act(h0, h1);   // (saturating conversion)
          }
          __syncwarp();
          const uint32_t sa = smem_u32(stg_base);
          stmatrix_x4_trans(sa + frag_off32, h[0], h[1], h[2], h[3]);          // token groups 0, 1 (features 0-7 | 8-15 each)
          stmatrix_x4_trans(sa + frag_off32 + 512, h[4], h[5], h[6], h[7]);    // token groups 2, 3
          __syncwarp();
          act_t* dst = st_ptr + static_cast<size_t>(c0) * p.out_ld_tok;
          const int n_ok = p.T - c0 - st_tok;
#pragma unroll
          for (int j = 0; j < 2; ++j)
            if (st_ok && 16 * j < n_ok)
              *reinterpret_cast<uint4*>(dst + static_cast<size_t>(16 * j) * p.out_ld_tok) = lds128(sa + rb_off32 + j * 512);
        } else if (p.stg_bytes >= 4096) {
          // fp32 (stream-K partial [slot][token][128 features] or the fp32 output): one 32-token box per chunk (4 KB
          // staging buffers) or two 16-token boxes (2 KB)
          stage_free();
          float* sb = reinterpret_cast<float*>(stg);
#pragma unroll
          for (int j = 0; j < 32; ++j) sb[j * 32 + lane] = v[j];
          if (contributor) stage_store(&map_part, quad * 32, c0, my_slot);
          else stage_store(&map_out, f0, mid, p.tok0 + c0);
        } else {
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            if (hh * 16 < cw) {
              stage_free();
              float* sb = reinterpret_cast<float*>(stg);
#pragma unroll
              for (int j = 0; j < 16; ++j) sb[j * 32 + lane] = v[hh * 16 + j];
              if (contributor) stage_store(&map_part, quad * 32, c0 + hh * 16, my_slot);
              else stage_store(&map_out, f0, mid, p.tok0 + c0 + hh * 16);
            }
          }
        }
      };
      // (everything above is address arithmetic: done while the MMAs of this piece are still running)
      if (has_mma) mbar_wait(&tmem_full_bar, acc_phase);
      tc_fence_after();
      for (int b0 = 0; b0 < n_pad && b0 < p.T; b0 += blk_cols) {
        const int b1 = min(b0 + blk_cols, n_pad);
        float v[32];
        if (frag && n_groups <= 1) {
          // software pipeline over this warp's chunks: the TMEM load of chunk i + 1 is in flight while chunk i is
          // converted and stored (two register sets, the loop is unrolled by two so that each keeps its registers)
          float vb[32];
          if (n_groups == 1) {
            load_group(0, n_contrib, b0, b1);
          }
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
          auto step = [&](int c0, float* cur, float* nxt) {
            tmem_ld_wait();
            const int cn = c0 + GEMM_BLK;
            if (cn < b1 && cn < p.T) issue(cn, nxt);
            if (n_groups == 1) add_fix(n_contrib, b0, b1, c0, cur);
            finish_chunk(c0, 32, cur);
          };
          int c0 = b0 + 32 * par;
          if (c0 < b1 && c0 < p.T) issue(c0, v);
          while (c0 < b1 && c0 < p.T) {
            step(c0, v, vb);
            c0 += GEMM_BLK;
            if (!(c0 < b1 && c0 < p.T)) break;
            step(c0, vb, v);
            c0 += GEMM_BLK;
          }
        } else if (n_groups <= 1) {
          if (n_groups == 1) {
            load_group(0, n_contrib, b0, b1);
          }
          for (int c0 = b0 + 32 * par; c0 < b1 && c0 < p.T; c0 += GEMM_BLK) {
            const int cw = min(32, b1 - c0);
            load_acc(c0, cw, v);
            if (n_groups == 1) add_fix(n_contrib, b0, b1, c0, v);
            finish_chunk(c0, cw, v);
          }
        } else {  // 64-column block: at most one chunk per warp; every warp takes part in every group load
          const int c0 = b0 + 32 * par;
          const bool has = c0 < b1 && c0 < p.T;
          const int cw = min(32, b1 - c0);
          if (has) load_acc(c0, cw, v);
          for (int g0 = 0; g0 < n_contrib; g0 += grp) {
            const int cnt = min(grp, n_contrib - g0);
            load_group(g0, cnt, b0, b1);
            if (has) add_fix(cnt, b0, b1, c0, v);
          }
          if (has) finish_chunk(c0, cw, v);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0 && has_mma) { if (mma2) mbar_arrive_leader(&tmem_empty_bar); else mbar_arrive(&tmem_empty_bar); }
      if (contributor) {
        if (lane == 0) { bulk_wait<0>(); fence_proxy_async_all(); }  // this warp's partial stores are complete
        __syncwarp();
        __threadfence();
        AF_EPI_BAR();
        if (etid == 0) {
          __threadfence();
          atomicExch(p.flags + my_slot, 1);
        }
      }
      ++piece;
      if (has_mma) acc_phase ^= 1;
    }
    if (lane == 0) bulk_wait<0>();  // all output stores are complete before the CTA exits
  }
#undef stg

  tc_fence_before();
  __syncthreads();
  if (p.cluster > 1) cluster_sync();  // no CTA leaves while its peer may still signal its barriers
  if (warp == GEMM_EPI_WARPS + 1) {
    tc_fence_after();
    if (mma2) tmem_dealloc_cg2(tmem_base, GEMM_TMEM_COLS); else tmem_dealloc(tmem_base, GEMM_TMEM_COLS);
  }
}
