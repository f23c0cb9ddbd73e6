// lmhead_sample.cuh - S8 of the default sampling path: the LM head as ONE persistent tcgen05 kernel whose epilogue reduces the
// sampling statistics, so the logits never reach HBM (BASELINE.json north_star (e) + (g)).
// Included by gemm_tcgen05.cuh between its device part (PTX wrappers, descriptors, TcMaps / TcGemmArgs) and its host part.
//
// Same swap-AB weight streamer as gemm_tcgen05_kernel (128 vocabulary ids = UMMA M = TMEM lanes, emitting rows = UMMA N), but:
//   * one CTA per SM walks a static list of (weight tile, model) units - unit u = blockIdx.x, + gridDim.x, ... - with its barriers,
//     tensor memory and the 192 KB ring set up once, so the weight stream never drains between tiles;
//   * the CTA owns all 512 TMEM columns = TWO accumulators of up to 256 token rows: while the sixteen epilogue warps reduce tile i
//     (Philox uniforms, Gumbel-max, max / sum exp - ALU work the one-tile-per-CTA kernel could not hide: 366 us against 265 us for the
//     plain LM head), the MMA warp already accumulates tile i + 1 in the other one.
// Per (tile, emitting row) the epilogue writes (max z, sum exp((z - max) / T), raw argmax, Gumbel-max value / id / z): out[row][tile][8]
// fp32; sample_merge_emit_kernel merges the tiles of a row in a fixed order. Results do not depend on which CTA owned a tile.

// ---- 16 token columns per lane (lane = vocabulary id), reduced across the 32 lanes of a warp by recursive halving - after four
// exchange rounds a lane holds ONE column reduced over 16 lanes, a fifth round finishes it: 16 shuffles per quantity instead of 80.
// The column a lane ends up with is lane >> 1. The combination tree is fixed: results are deterministic.
template <typename Op>
__device__ __forceinline__ float tc_reduce16(float (&a)[16], int lane, Op op) {
  bool hi = lane & 16;
#pragma unroll
  for (int i = 0; i < 8; ++i) { const float send = hi ? a[i] : a[i + 8], keep = hi ? a[i + 8] : a[i]; a[i] = op(keep, __shfl_xor_sync(0xffffffffu, send, 16)); }
  hi = lane & 8;
#pragma unroll
  for (int i = 0; i < 4; ++i) { const float send = hi ? a[i] : a[i + 4], keep = hi ? a[i + 4] : a[i]; a[i] = op(keep, __shfl_xor_sync(0xffffffffu, send, 8)); }
  hi = lane & 4;
#pragma unroll
  for (int i = 0; i < 2; ++i) { const float send = hi ? a[i] : a[i + 2], keep = hi ? a[i + 2] : a[i]; a[i] = op(keep, __shfl_xor_sync(0xffffffffu, send, 4)); }
  hi = lane & 2;
  { const float send = hi ? a[0] : a[1], keep = hi ? a[1] : a[0]; a[0] = op(keep, __shfl_xor_sync(0xffffffffu, send, 2)); }
  return op(a[0], __shfl_xor_sync(0xffffffffu, a[0], 1));
}

constexpr int kLmTmemCols = 512;       // two accumulators of kTcMaxRows columns
constexpr int kLmRingBytes = 192 * 1024;
constexpr int kLmEpiWarps = 16;        // four per TMEM lane quarter: the epilogue's dependent chains (shuffle trees, Philox rounds) are latency-bound
constexpr int kLmThreads = (3 + kLmEpiWarps) * 32;   // warps 0 weight TMA, 1 MMA, 6 activation TMA; 2-5, 7-10, 11-14, 15-18 epilogue
constexpr int kLmExtraBytes = 2048 + (kLmEpiWarps / 4) * 2 * 4 * 16 * 6 * 4;   // (t, seq_id) of a chunk's rows + per-part double-buffered quarter partials
constexpr int kLmSmemBytes = kLmRingBytes + kLmExtraBytes + 1024;

__global__ void __launch_bounds__(kLmThreads, 1)
lmhead_sample_kernel(const __grid_constant__ TcMaps maps, const __grid_constant__ Pair<TcGemmArgs> gp) {
  extern __shared__ uint8_t lm_smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * kTcMaxStages + 4];
  __shared__ uint32_t tmem_base_smem;

  pdl_trigger();
  // emitting rows of the two models: scheduler output, complete before any kernel of the chain starts
  const int rows_of[2] = {gp.m[0].rows_ptr ? *gp.m[0].rows_ptr : gp.m[0].rows_fixed, gp.m[1].rows_ptr ? *gp.m[1].rows_ptr : gp.m[1].rows_fixed};
  const int n_act = (rows_of[0] > 0 ? 1 : 0) + (rows_of[1] > 0 ? 1 : 0);
  const int N = gp.m[0].N, K = gp.m[0].K;
  const int tiles = (N + kTcTileN - 1) / kTcTileN;
  const int n_units = tiles * n_act;                       // models interleaved: both finish together
  if ((int)blockIdx.x >= n_units) { pdl_wait(); return; }  // includes "nothing emits this step"
  const int only = rows_of[0] > 0 ? 0 : 1;
  auto unit_model = [&](int u) { return n_act == 2 ? (u & 1) : only; };
  auto unit_tile = [&](int u) { return n_act == 2 ? (u >> 1) : u; };
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int kb_total = (K + kTcBlockK - 1) / kTcBlockK;
  auto chunk_cols = [&](int rows, int r0) { return ((min(rows - r0, kTcMaxRows) + kTcRowBox - 1) / kTcRowBox) * kTcRowBox; };
  // one stage layout for both models: the larger first chunk decides
  const int nbox_max = max(rows_of[0] > 0 ? chunk_cols(rows_of[0], 0) : 0, rows_of[1] > 0 ? chunk_cols(rows_of[1], 0) : 0) / kTcRowBox;
  const int stage_bytes = kTcWBytes + nbox_max * kTcABoxBytes;
  const int n_stages = min(kTcMaxStages, kLmRingBytes / stage_bytes);

  const uint32_t ring = (ptx::smem_u32(lm_smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (uint32_t)(kTcMaxStages + s); };
  auto acc_full_bar = [&](int b) { return bar0 + 8u * (uint32_t)(2 * kTcMaxStages + b); };
  auto acc_empty_bar = [&](int b) { return bar0 + 8u * (uint32_t)(2 * kTcMaxStages + 2 + b); };

  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { ptx::mbar_init(full_bar(s), 2); ptx::mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(acc_full_bar(b), 1); ptx::mbar_init(acc_empty_bar(b), kLmEpiWarps); }
    ptx::fence_mbar_init();
    ptx::prefetch_tmap(&maps.w[0]); ptx::prefetch_tmap(&maps.w[1]);
    ptx::prefetch_tmap(maps.a[0]); ptx::prefetch_tmap(maps.a[1]);
  }
  if (warp == 2) ptx::tmem_alloc<kLmTmemCols>(ptx::smem_u32(&tmem_base_smem));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  if (warp == 0) {
    // ===== weight producer: never waits for the predecessor kernel; runs ahead across tiles as far as the ring allows
    const uint64_t pol_w = ptx::policy_evict_first();
    int it = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const int mdl = unit_model(u), n0 = unit_tile(u) * kTcTileN;
      const int n_chunks = (rows_of[mdl] + kTcMaxRows - 1) / kTcMaxRows;
      for (int c = 0; c < n_chunks; ++c)
        for (int kb = 0; kb < kb_total; ++kb, ++it) {
          const int s = it % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(it / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)kTcWBytes);
            ptx::tma_load_2d(ring + (uint32_t)(s * stage_bytes), &maps.w[mdl], kb * kTcBlockK, n0, full_bar(s), pol_w);
          }
          __syncwarp();
        }
    }
  } else if (warp == 6) {
    // ===== activation producer: the final-norm rows of the emitting sequences (L2 evict-last), greedy 128/64/32/16-row boxes
    const uint64_t pol_a = ptx::policy_evict_last();
    pdl_wait();
    int it = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const int mdl = unit_model(u), rows = rows_of[mdl];
      const CUtensorMap* tmap_a = maps.a[mdl];
      const int n_chunks = (rows + kTcMaxRows - 1) / kTcMaxRows;
      for (int c = 0; c < n_chunks; ++c) {
        const int nbox = chunk_cols(rows, c * kTcMaxRows) / kTcRowBox, r0 = c * kTcMaxRows;
        for (int kb = 0; kb < kb_total; ++kb, ++it) {
          const int s = it % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(it / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)(nbox * kTcABoxBytes));
            const uint32_t dst = ring + (uint32_t)(s * stage_bytes) + kTcWBytes;
            int j = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              const int bx = 8 >> b;
              while (nbox - j >= bx) {
                ptx::tma_load_2d(dst + j * kTcABoxBytes, tmap_a + b, kb * kTcBlockK, r0 + j * kTcRowBox, full_bar(s), pol_a);
                j += bx;
              }
            }
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: pass ci (a tile's chunk) accumulates in accumulator ci & 1
    int it = 0, ci = 0;
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const int rows = rows_of[unit_model(u)];
      const int n_chunks = (rows + kTcMaxRows - 1) / kTcMaxRows;
      for (int c = 0; c < n_chunks; ++c, ++ci) {
        const uint32_t idesc = umma_idesc_bf16(chunk_cols(rows, c * kTcMaxRows));
        const uint32_t acc = tmem_base + (uint32_t)((ci & 1) * kTcMaxRows);
        ptx::mbar_wait(acc_empty_bar(ci & 1), ((uint32_t)(ci >> 1) & 1u) ^ 1u);
        ptx::tc_fence_after();
        for (int kb = 0; kb < kb_total; ++kb, ++it) {
          const int s = it % n_stages;
          ptx::mbar_wait(full_bar(s), (uint32_t)(it / n_stages) & 1u);
          ptx::tc_fence_after();
          const uint32_t sw = ring + (uint32_t)(s * stage_bytes);
          const uint64_t dw = umma_desc_sw128(sw), da = umma_desc_sw128(sw + kTcWBytes);
          if (ptx::elect_one()) {
#pragma unroll
            for (int k = 0; k < kTcBlockK / 16; ++k)
              ptx::umma_bf16(acc, dw + (uint64_t)(2 * k), da + (uint64_t)(2 * k), idesc, (kb > 0 || k > 0) ? 1u : 0u);
            ptx::umma_commit(empty_bar(s));
          }
          __syncwarp();
        }
        if (ptx::elect_one()) ptx::umma_commit(acc_full_bar(ci & 1));
        __syncwarp();
      }
    }
  } else {
    // ===== epilogue: warp w may touch TMEM lanes 32*(w%4)..+31; lane = vocabulary id n, column = emitting row; 16 columns at a time;
    // the four warps of a lane quarter ("parts") take every fourth 16-column group; the four quarters of a part are combined through
    // shared memory into ONE partial per (tile, row)
    const int q = warp & 3;
    const int part = warp < 6 ? 0 : (warp - 3) >> 2;          // warps 2-5: 0, 7-10: 1, 11-14: 2, 15-18: 3
    uint8_t* extra = lm_smem_raw + (ring - ptx::smem_u32(lm_smem_raw)) + kLmRingBytes;
    int* s_t = reinterpret_cast<int*>(extra);                 // [256] t = index of the token being emitted by the row's sequence
    int* s_sid = s_t + kTcMaxRows;                            // [256] its sequence id
    float* s_part = reinterpret_cast<float*>(extra + 2048);   // [part 4][buffer 2][quarter 4][16 columns][6]
    const int et = (warp >= 7 ? warp - 3 : warp - 2) * 32 + lane;   // 0..511 over the sixteen epilogue warps
    int ci = 0, it16 = 0, loaded = -1;                        // it16 runs on across passes: the partial buffers keep alternating
    pdl_wait();                                               // the predecessor may still be reading the buffer this kernel writes
    for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
      const int mdl = unit_model(u), tile = unit_tile(u), n0 = tile * kTcTileN;
      const TcGemmArgs& g = gp.m[mdl];
      const int rows = rows_of[mdl];
      const int n = n0 + q * 32 + lane;
      const bool n_ok = n < N;
      const float inv_t = g.inv_t;
      const int n_chunks = (rows + kTcMaxRows - 1) / kTcMaxRows;
      for (int c = 0; c < n_chunks; ++c, ++ci) {
        const int r0 = c * kTcMaxRows;
        const int crow = min(rows - r0, kTcMaxRows);
        if (loaded != mdl * 65536 + c) {                      // (t, seq_id) of this (model, chunk)'s rows; unchanged from tile to tile
          ptx::bar_sync_id<1>(kLmEpiWarps * 32);              // the previous pass's readers are done
          if (et < kTcMaxRows) {
            const int j = r0 + et;
            const int slot = j < rows ? g.emit_slot[j] : 0;
            s_t[et] = j < rows ? g.n_emit[slot] + 1 : 0;
            s_sid[et] = j < rows ? g.seq_id[slot] : 0;
          }
          ptx::bar_sync_id<1>(kLmEpiWarps * 32);
          loaded = mdl * 65536 + c;
        }
        const uint32_t acc = tmem_base + (uint32_t)((ci & 1) * kTcMaxRows);
        ptx::mbar_wait(acc_full_bar(ci & 1), (uint32_t)(ci >> 1) & 1u);
        ptx::tc_fence_after();
        for (int c0 = 16 * part; c0 < crow; c0 += 16 * (kLmEpiWarps / 4), ++it16) {
          uint32_t v[16];
          ptx::tmem_ld16(acc + ((uint32_t)(q * 32) << 16) + (uint32_t)c0, v);
          ptx::tmem_ld_wait();
          float z[16], w[16];
#pragma unroll
          for (int k = 0; k < 16; ++k) { z[k] = (n_ok && c0 + k < crow) ? __uint_as_float(v[k]) : -INFINITY; w[k] = z[k]; }
          // column maxima of z, then known to every lane
          const float mine_m = tc_reduce16(w, lane, [](float x, float y) { return fmaxf(x, y); });
          float M[16];
#pragma unroll
          for (int k = 0; k < 16; ++k) M[k] = __shfl_sync(0xffffffffu, mine_m, 2 * k);
          // raw argmax: the lowest lane (= lowest id) that holds the maximum; sum of exp((z - max) / T)
          int my_raw = 0;
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            const unsigned b = __ballot_sync(0xffffffffu, z[k] == M[k] && z[k] != -INFINITY);
            if (k == (lane >> 1)) my_raw = b ? __ffs(b) - 1 : 0;
            w[k] = z[k] == -INFINITY ? 0.f : expf((z[k] - M[k]) * inv_t);
          }
          const float mine_s = tc_reduce16(w, lane, [](float x, float y) { return x + y; });
          // Gumbel-max: g = -ln(-log1p(-u)), u from Philox-4x32-10 at counter (n >> 2, t, seq_id, 0), word n & 3 - the block of four ids is
          // computed by the lane whose (lane & 3) equals (column & 3) and handed to its three neighbours
          float mine_gv = -INFINITY, mine_gz = 0.f; int my_g = 0;
          if (!g.greedy) {
            uint32_t blk[4][4];
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              const int k = 4 * kk + (lane & 3);
              blk[kk][0] = (uint32_t)(n >> 2); blk[kk][1] = (uint32_t)s_t[c0 + k]; blk[kk][2] = (uint32_t)s_sid[c0 + k]; blk[kk][3] = 0u;
              philox4x32_10(blk[kk], g.key0, g.key1);
            }
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              const int src = (lane & ~3) | (k & 3);
              const uint32_t w0 = __shfl_sync(0xffffffffu, blk[k >> 2][0], src), w1 = __shfl_sync(0xffffffffu, blk[k >> 2][1], src);
              const uint32_t w2 = __shfl_sync(0xffffffffu, blk[k >> 2][2], src), w3 = __shfl_sync(0xffffffffu, blk[k >> 2][3], src);
              const uint32_t r = (lane & 2) ? ((lane & 1) ? w3 : w2) : ((lane & 1) ? w1 : w0);
              w[k] = z[k] == -INFINITY ? -INFINITY : z[k] * inv_t + gumbel_from_uniform(uniform_from_bits(r));
            }
            float gg[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) gg[k] = w[k];
            mine_gv = tc_reduce16(w, lane, [](float x, float y) { return fmaxf(x, y); });
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              const float Gk = __shfl_sync(0xffffffffu, mine_gv, 2 * k);
              const unsigned b = __ballot_sync(0xffffffffu, gg[k] == Gk && gg[k] != -INFINITY);
              const int wl = b ? __ffs(b) - 1 : 0;
              const float zw = __shfl_sync(0xffffffffu, z[k], wl);
              if (k == (lane >> 1)) { my_g = wl; mine_gz = zw; }
            }
          }
          // this quarter's partial of column lane >> 1 -> shared memory; four quarters -> one partial per (tile, row)
          float* sp = s_part + ((size_t)(part * 2 + (it16 & 1)) * 4 + q) * 16 * 6;
          if ((lane & 1) == 0) {
            float* e = sp + (lane >> 1) * 6;
            e[0] = mine_m; e[1] = mine_s; e[2] = __int_as_float(n0 + q * 32 + my_raw); e[3] = mine_gv; e[4] = __int_as_float(n0 + q * 32 + my_g); e[5] = mine_gz;
          }
          if (part == 0) ptx::bar_sync_id<2>(128); else if (part == 1) ptx::bar_sync_id<3>(128); else if (part == 2) ptx::bar_sync_id<4>(128); else ptx::bar_sync_id<5>(128);
          if (q == 0 && lane < 16 && c0 + lane < crow) {
            const float* e0 = s_part + ((size_t)(part * 2 + (it16 & 1)) * 4) * 16 * 6 + lane * 6;
            SamplePart a{e0[0], e0[1], e0[3], e0[5], __float_as_int(e0[2]), __float_as_int(e0[4])};
#pragma unroll
            for (int qq = 1; qq < 4; ++qq) {
              const float* e = e0 + qq * 16 * 6;
              sample_part_merge(a, SamplePart{e[0], e[1], e[3], e[5], __float_as_int(e[2]), __float_as_int(e[4])}, inv_t);
            }
            float4* dst = reinterpret_cast<float4*>(g.out + ((size_t)(r0 + c0 + lane) * tiles + tile) * kTcSampleVals);   // [row][tile][8]
            dst[0] = make_float4(a.m, a.s, __int_as_float(a.raw_id), a.gv);
            dst[1] = make_float4(__int_as_float(a.g_id), a.gz, 0.f, 0.f);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(acc_empty_bar(ci & 1));
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<kLmTmemCols>(tmem_base);
}
