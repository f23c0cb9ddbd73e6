// gemm_streamk.cuh - S7's gate/up projection + SwiGLU at decode row counts as ONE persistent, exactly balanced kernel for both models
// (BASELINE.json north_star (e)).
//
// Why: at ~128 token rows per model the one-tile-per-CTA kernel (gemm_tcgen05.cuh) is bound by what an SM can pull through TMA, not
// by HBM - every 128-row weight tile (16 KB per k-block) drags the whole activation tile (18 KB at 144 rows) out of L2 again - and
// its 304 tiles do not fit the 296 CTA slots (profiles/gemm_sweep_r1.md, profiles/gemm_r2.md: 3.6 TB/s, SMs active 62% of the launch).
// Here
//   * a unit is a PAIR of adjacent 128-row weight tiles sharing every activation stage (one 256-row TMA box, two M = 128 accumulators):
//     half the activation bytes per weight byte;
//   * NR = SMs / 2 CTAs serve a model. Its DT tile pairs are dealt as Wp = DT / NR WHOLE pairs per CTA (pair r, r + NR, ...: the whole
//     K range in one accumulator, plain SwiGLU epilogue) and the L = DT - Wp NR LEFTOVER pairs are split along K into S = NR / L slices
//     each, one slice per CTA (the split-K remainder of a stream-K schedule, with every other cut on a pair boundary).
//     Every SM streams the same bytes (4B shape: 40 + 40/37 k-blocks of 76 pairs on 74 CTAs), with one set of barriers, one ring and
//     no drain between the pieces;
//   * a CTA computes its slice FIRST, leaves the fp32 partial in scratch memory and counts itself in; then, while its whole pairs
//     stream, its epilogue warps reduce a 1/S share of the leftover pair - all S partials in slice order - and apply SwiGLU. The
//     cross-CTA hand-over is over in the first microseconds of the launch and never sits on the critical path. (A first version cut
//     the k-block sequence into equal contiguous ranges and let the owner of a pair's first k-block add its neighbour's partial in the
//     LAST epilogue: two dependent L2 round trips of ~3 us each under a saturated memory system, exposed at the end - 63 us, no gain.)
// The cuts are a function of (N, K, SM count) only: every output is the same sum in the same order whatever the batch holds - results
// stay independent of the batch, of the step's row count and of which models are active. One model active (solo decoding, the first
// prefill): range r is served by CTAs r and r + NR, one 128-row tile of every pair each, same k-ranges. More than 256 token rows:
// chunks of 256 in the OUTER loop (weights re-streamed per chunk, as in the one-tile kernel); the scratch is one chunk deep and the
// arrival counters run on across chunks.
//   warp 0: weight TMA   warp 6: activation TMA   warp 1: MMA issuer   warps 2-5, 7-18: epilogue + the leftover reduction
#pragma once
#include "gemm_tcgen05.cuh"

namespace tandem {

constexpr int kSkEpiWarps = 16;         // four per TMEM lane quarter: the SwiGLU epilogue of the last pair is exposed, and it is issue-latency bound
constexpr int kSkThreads = (3 + kSkEpiWarps) * 32;
constexpr int kSkMaxStages = 8;
constexpr int kSkRingBytes = 208 * 1024;
constexpr int kSkSmemBytes = kSkRingBytes + 1024;
constexpr int kSkPairRows = 2 * kTcTileN;
constexpr long long kSkSpinLimit = 4000000000ll;   // ~2 s of SM clocks: a wait this long means a lost signal - flag it and go on, never hang the GPU

// DT tile pairs, KB k-blocks, NR CTAs per model, Wp whole pairs per CTA, L leftover pairs in S k-slices each (S = 0: none)
struct SkGeo { int DT, KB, NR, Wp, L, S; };
__host__ __device__ __forceinline__ SkGeo sk_geo(int N, int K, int n_ctas) {
  SkGeo g;
  g.DT = (N + kSkPairRows - 1) / kSkPairRows; g.KB = (K + kTcBlockK - 1) / kTcBlockK; g.NR = n_ctas / 2;
  g.Wp = g.NR > 0 ? g.DT / g.NR : 0; g.L = g.DT - g.Wp * g.NR;
  g.S = g.L > 0 ? g.NR / g.L : 0;
  if (g.S > g.KB) g.S = g.KB;          // every slice holds at least one k-block
  return g;
}
// served when every CTA owns at least one whole pair (the leftovers are then a small remainder)
inline bool sk_applicable(int N, int K, int n_sms) {
  if (n_sms < 2 || (N & 1) || (K % 8)) return false;
  const SkGeo g = sk_geo(N, K, n_sms);
  return g.Wp >= 1;
}

struct SkMaps { CUtensorMap w256[2], w128[2], a[2][4]; };   // per model: weight boxes of 256 / 128 rows; activation boxes of 128/64/32/16 rows
struct SkArgs {
  const int32_t* rows_ptr[2];   // live token rows of each model (device)
  bf16* act_out[2];             // [rows, N/2] silu(gate) * up; W rows interleaved 2i = gate_i, 2i+1 = up_i
  int N, K;
  float* scratch;               // [2 models][NR slices in (leftover pair, slice) order][2 tiles][128 weight rows][scratch_rows] fp32 partials
  int scratch_rows;             // >= min(256, row capacity), multiple of 32
  int32_t* arrived;             // [2][NR] per (model, leftover pair): partials written so far, cumulative over the chunks of a launch
  int32_t* reduced;             // [2][NR] per (model, leftover pair): reducers finished so far; the last one returns both counters to 0
  int32_t* fault;               // raised (1) when a bounded wait expired: results invalid (mapped host word)
};

namespace ptx {
__device__ __forceinline__ int ld_acquire_gpu(const int32_t* p) { int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v; }
}  // namespace ptx

// Bounded spin on a counter advanced by other CTAs of this launch (all CTAs are co-resident: grid <= SM count, one CTA per SM).
__device__ __forceinline__ void sk_spin_ge(const int32_t* p, int target, int32_t* fault) {
  const long long t0 = clock64();
  int it = 0;
  while (ptx::ld_acquire_gpu(p) < target) {
    if ((++it & 1023) == 0 && clock64() - t0 > kSkSpinLimit) { *fault = 1; break; }
  }
}

__global__ void __launch_bounds__(kSkThreads, 1)
gateup_streamk_kernel(const __grid_constant__ SkMaps maps, const __grid_constant__ SkArgs a) {
  extern __shared__ uint8_t sk_smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * kSkMaxStages + 4];
  __shared__ uint32_t tmem_base_smem;

  pdl_trigger();
  const int R0 = *a.rows_ptr[0], R1 = *a.rows_ptr[1];       // scheduler output: complete before any kernel of the chain starts
  const int cta = blockIdx.x;
  const SkGeo g = sk_geo(a.N, a.K, gridDim.x);
  if (R0 + R1 <= 0 || cta >= 2 * g.NR) { pdl_wait(); return; }   // uniform over the grid / the odd CTA of an odd SM count
  const bool both = R0 > 0 && R1 > 0;
  const int mdl = both ? cta / g.NR : (R0 > 0 ? 0 : 1);
  const int half = both ? 0 : cta / g.NR;                   // one model active: which 128-row tile of every pair this CTA takes
  const int r = cta % g.NR;
  const int rows = mdl ? R1 : R0;
  const int ntile = both ? 2 : 1;
  const int KB = g.KB;
  // this CTA's slice of a leftover pair (computed first), then its whole pairs
  const bool has_slice = g.S > 0 && r < g.L * g.S;
  const int lp = has_slice ? r / g.S : 0, sj = has_slice ? r - lp * g.S : 0;
  const int sk0 = has_slice ? KB * sj / g.S : 0, sk1 = has_slice ? KB * (sj + 1) / g.S : 0;
  const int n_pieces = (has_slice ? 1 : 0) + g.Wp;
  const int n_chunks = (rows + kTcMaxRows - 1) / kTcMaxRows;
  auto chunk_cols = [&](int r0) { return ((min(rows - r0, kTcMaxRows) + kTcRowBox - 1) / kTcRowBox) * kTcRowBox; };
  const int ncols_max = chunk_cols(0);
  const int wbytes = ntile * kTcWBytes;
  const int stage_bytes = wbytes + (ncols_max / kTcRowBox) * kTcABoxBytes;
  const int n_stages = min(kSkMaxStages, kSkRingBytes / stage_bytes);
  // accumulators: a piece needs ntile * tile_cols columns; two buffers of 256 columns when that fits (<= 128 token rows, or one tile), else one of 512
  const uint32_t tile_cols = ncols_max > 128 ? 256u : 128u;
  const int nbuf = (uint32_t)ntile * tile_cols <= 256u ? 2 : 1;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  const uint32_t ring = (ptx::smem_u32(sk_smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (uint32_t)(kSkMaxStages + s); };
  auto acc_full_bar = [&](int b) { return bar0 + 8u * (uint32_t)(2 * kSkMaxStages + b); };
  auto acc_empty_bar = [&](int b) { return bar0 + 8u * (uint32_t)(2 * kSkMaxStages + 2 + b); };
  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { ptx::mbar_init(full_bar(s), 2); ptx::mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(acc_full_bar(b), 1); ptx::mbar_init(acc_empty_bar(b), kSkEpiWarps); }
    ptx::fence_mbar_init();
    ptx::prefetch_tmap(both ? &maps.w256[mdl] : &maps.w128[mdl]);
    ptx::prefetch_tmap(maps.a[mdl]);
  }
  if (warp == 2) ptx::tmem_alloc<512>(ptx::smem_u32(&tmem_base_smem));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  // Every role walks the same sequence: for each 256-row chunk, piece 0 = the slice (if any), then the whole pairs r, r + NR, ...
  // piece pc -> (tile pair t, k-blocks [k0, k1))
  auto piece = [&](int pc, int& t, int& k0, int& k1) {
    if (has_slice && pc == 0) { t = g.Wp * g.NR + lp; k0 = sk0; k1 = sk1; }
    else { t = r + (has_slice ? pc - 1 : pc) * g.NR; k0 = 0; k1 = KB; }
  };

  if (warp == 0) {
    // ===== weight producer: weights depend on nothing - it never waits for the predecessor kernel and runs ahead across pieces
    const uint64_t pol_w = ptx::policy_evict_first();
    const CUtensorMap* mw = both ? &maps.w256[mdl] : &maps.w128[mdl];
    int n = 0;
    for (int ch = 0; ch < n_chunks; ++ch)
      for (int pc = 0; pc < n_pieces; ++pc) {
        int t, k0, k1; piece(pc, t, k0, k1);
        const int n0 = t * kSkPairRows + half * kTcTileN;
        for (int kb = k0; kb < k1; ++kb, ++n) {
          const int s = n % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(n / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)wbytes);
            ptx::tma_load_2d(ring + (uint32_t)(s * stage_bytes), mw, kb * kTcBlockK, n0, full_bar(s), pol_w);
          }
          __syncwarp();
        }
      }
  } else if (warp == 6) {
    // ===== activation producer (L2 evict-last): greedy 128/64/32/16-row boxes
    const uint64_t pol_a = ptx::policy_evict_last();
    const CUtensorMap* ma = maps.a[mdl];
    pdl_wait();                                            // the activations come from the predecessor kernel
    int n = 0;
    for (int ch = 0; ch < n_chunks; ++ch) {
      const int r0 = ch * kTcMaxRows, nbox = chunk_cols(r0) / kTcRowBox;
      for (int pc = 0; pc < n_pieces; ++pc) {
        int t, k0, k1; piece(pc, t, k0, k1);
        for (int kb = k0; kb < k1; ++kb, ++n) {
          const int s = n % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(n / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)(nbox * kTcABoxBytes));
            const uint32_t dst = ring + (uint32_t)(s * stage_bytes) + (uint32_t)wbytes;
            int j = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              const int bx = 8 >> b;
              while (nbox - j >= bx) { ptx::tma_load_2d(dst + j * kTcABoxBytes, ma + b, kb * kTcBlockK, r0 + j * kTcRowBox, full_bar(s), pol_a); j += bx; }
            }
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: piece i accumulates in buffer i & 1 (when two fit)
    int n = 0, i = 0;
    for (int ch = 0; ch < n_chunks; ++ch) {
      const uint32_t idesc = umma_idesc_bf16(chunk_cols(ch * kTcMaxRows));
      for (int pc = 0; pc < n_pieces; ++pc, ++i) {
        int t, k0, k1; piece(pc, t, k0, k1);
        const int buf = nbuf == 2 ? (i & 1) : 0, use = nbuf == 2 ? (i >> 1) : i;
        const uint32_t acc = tmem_base + (uint32_t)buf * 256u;
        ptx::mbar_wait(acc_empty_bar(buf), ((uint32_t)use & 1u) ^ 1u);
        ptx::tc_fence_after();
        for (int kb = k0; kb < k1; ++kb, ++n) {
          const int s = n % n_stages;
          ptx::mbar_wait(full_bar(s), (uint32_t)(n / n_stages) & 1u);
          ptx::tc_fence_after();
          const uint32_t sw = ring + (uint32_t)(s * stage_bytes);
          const uint64_t da = umma_desc_sw128(sw + (uint32_t)wbytes);
          if (ptx::elect_one()) {
            for (int j = 0; j < ntile; ++j) {
              const uint64_t dw = umma_desc_sw128(sw + (uint32_t)(j * kTcWBytes));
#pragma unroll
              for (int k = 0; k < kTcBlockK / 16; ++k)
                ptx::umma_bf16(acc + (uint32_t)j * tile_cols, dw + (uint64_t)(2 * k), da + (uint64_t)(2 * k), idesc, (kb > k0 || k > 0) ? 1u : 0u);
            }
            ptx::umma_commit(empty_bar(s));
          }
          __syncwarp();
        }
        if (ptx::elect_one()) ptx::umma_commit(acc_full_bar(buf));
        __syncwarp();
      }
    }
  } else {
    // ===== epilogue: warp w may touch TMEM lanes 32*(w%4)..+31; lane = weight row, column = token row; sixteen warps = four per lane
    // quarter ("parts"). Tile pairs: part & 1 = tile, part >> 1 = which of every two 32-column groups; a single tile: every fourth group.
    const int q = warp & 3;
    const int part = warp < 6 ? 0 : (warp - 3) >> 2;       // warps 2-5: 0, 7-10: 1, 11-14: 2, 15-18: 3
    const int tid_e = (warp >= 7 ? warp - 3 : warp - 2) * 32 + lane;
    const int j_tile = ntile == 2 ? (part & 1) : 0;
    const int c_first = ntile == 2 ? 32 * (part >> 1) : 32 * part, c_step = ntile == 2 ? 64 : 128;
    const int I = a.N >> 1;
    const size_t srows = (size_t)a.scratch_rows;           // multiple of 32
    const size_t blk = (size_t)kTcTileN * srows;           // floats of one (slice, tile) block: [weight row 128][scratch_rows]
    float* const pair_scr = a.scratch + ((size_t)mdl * g.NR + (size_t)lp * g.S) * 2 * blk;   // the S slices of leftover pair lp
    // a thread's 32 columns of a group are 128 contiguous bytes of its weight row
    float* my_part = pair_scr + ((size_t)sj * 2 + (ntile == 2 ? j_tile : half)) * blk + (size_t)(q * 32 + lane) * srows;
    int32_t* const arrived = a.arrived + mdl * g.NR + lp;
    int32_t* const reduced = a.reduced + mdl * g.NR + lp;
    const int per_chunk = g.S * (both ? 1 : 2);             // arrivals per chunk: one model active = two CTAs (tiles) per slice
    bf16* act = a.act_out[mdl];
    pdl_wait();                                            // the predecessor may still be reading the buffers this kernel writes
    int i = 0;
    for (int ch = 0; ch < n_chunks; ++ch) {
      const int r0 = ch * kTcMaxRows, crow = min(rows - r0, kTcMaxRows);
      for (int pc = 0; pc < n_pieces; ++pc, ++i) {
        int t, k0, k1; piece(pc, t, k0, k1);
        const int buf = nbuf == 2 ? (i & 1) : 0, use = nbuf == 2 ? (i >> 1) : i;
        const uint32_t acc = tmem_base + (uint32_t)buf * 256u + (uint32_t)j_tile * tile_cols + ((uint32_t)(q * 32) << 16);
        if (has_slice && pc == 0) {
          // ---- this CTA's k-slice of leftover pair lp: fp32 partial -> scratch, count in; then its share of the pair's reduction
          if (ch > 0) {                                    // the scratch is one chunk deep: every reducer must be done with the previous chunk
            if (lane == 0) sk_spin_ge(reduced, ch * g.S, a.fault);
            __syncwarp();
          }
          ptx::mbar_wait(acc_full_bar(buf), (uint32_t)use & 1u);
          ptx::tc_fence_after();
          for (int c0 = c_first; c0 < crow; c0 += c_step) {
            uint32_t v[32];
            ptx::tmem_ld32(acc + (uint32_t)c0, v);
            ptx::tmem_ld_wait();
            float4* dst = reinterpret_cast<float4*>(my_part + c0);
#pragma unroll
            for (int j = 0; j < 8; ++j)
              dst[j] = make_float4(__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]), __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3]));
          }
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(acc_empty_bar(buf));
          __threadfence();
          ptx::bar_sync_id<1>(kSkEpiWarps * 32);
          if (tid_e == 0) atomicAdd(arrived, 1);
          if (half == 0) {
            // reduce gate/up row pairs [rp0, rp1) of the leftover pair over its S slices, in slice order; thread = (row pair, token column)
            const int rp0 = kTcTileN * sj / g.S, rp1 = kTcTileN * (sj + 1) / g.S;
            if (lane == 0) sk_spin_ge(arrived, (ch + 1) * per_chunk, a.fault);
            __syncwarp();
            for (int idx = tid_e; idx < (rp1 - rp0) * crow; idx += kSkEpiWarps * 32) {
              const int rp = rp0 + idx / crow, c = idx - (idx / crow) * crow;
              const float* src = pair_scr + (size_t)(rp >> 6) * blk + (size_t)(2 * (rp & 63)) * srows + c;   // tile rp / 64, weight row 2 (rp % 64): gate; + srows: up
              float gate = 0.f, up = 0.f;
              for (int s = 0; s < g.S; ++s) { gate += __ldcg(src + (size_t)s * 2 * blk); up += __ldcg(src + (size_t)s * 2 * blk + srows); }
              const int ii = t * kTcTileN + rp;
              if (2 * ii < a.N) act[(size_t)(r0 + c) * I + ii] = __float2bfloat16_rn(__fdividef(gate, 1.f + __expf(-gate)) * up);
            }
            ptx::bar_sync_id<1>(kSkEpiWarps * 32);
            if (tid_e == 0) {
              const int done = atomicAdd(reduced, 1) + 1;
              if (done == n_chunks * g.S) { atomicExch(arrived, 0); atomicExch(reduced, 0); }   // the launch's last reducer: both counters back to 0
            }
          }
          continue;
        }
        // ---- a whole pair: SwiGLU on the complete sums
        const int n = t * kSkPairRows + half * kTcTileN + j_tile * kTcTileN + q * 32 + lane;   // weight row of this lane
        ptx::mbar_wait(acc_full_bar(buf), (uint32_t)use & 1u);
        ptx::tc_fence_after();
        for (int c0 = c_first; c0 < crow; c0 += c_step) {
          uint32_t v[32];
          ptx::tmem_ld32(acc + (uint32_t)c0, v);
          ptx::tmem_ld_wait();
          // even lane = gate row i, odd lane = up row i of the same intermediate index i: swap halves of the 32 columns so that the
          // even lane finishes columns [0,16) and the odd lane columns [16,32)
          const bool odd = lane & 1;
          bf16* dst = act + (size_t)(r0 + c0 + (odd ? 16 : 0)) * I + (n >> 1);
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const float mine = __uint_as_float(odd ? v[16 + j] : v[j]);
            const float send = __uint_as_float(odd ? v[j] : v[16 + j]);
            const float recv = __shfl_xor_sync(0xffffffffu, send, 1);
            const float gate = odd ? recv : mine, up = odd ? mine : recv;
            if (c0 + (odd ? 16 : 0) + j < crow && n < a.N) dst[(size_t)j * I] = __float2bfloat16_rn(__fdividef(gate, 1.f + __expf(-gate)) * up);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(acc_empty_bar(buf));
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<512>(tmem_base);
}

// Launch for both models. Returns 0, or -1 (TANDEM_EINVAL) / -3 (TANDEM_ECUDA).
inline int sk_gateup_launch(TcGemmPlans* p, const void* const* A, const void* const* W, int N, int K, void* const* act_out, const int32_t* const* rows_ptr,
                            int rows_cap, float* scratch, int scratch_rows, int32_t* arrived, int32_t* reduced, int32_t* fault, int n_sms, cudaStream_t s, bool pdl) {
  if (!p || !sk_applicable(N, K, n_sms)) return -1;
  SkMaps maps;
  SkArgs a;
  for (int m = 0; m < 2; ++m) {
    const CUtensorMap* w256 = tc_gemm_map(p, W[m], N, K, kSkPairRows);
    const CUtensorMap* w128 = tc_gemm_map(p, W[m], N, K, kTcTileN);
    if (!w256 || !w128) return -3;
    maps.w256[m] = *w256; maps.w128[m] = *w128;
    for (int b = 0; b < 4; ++b) {
      const CUtensorMap* ma = tc_gemm_map(p, A[m], rows_cap, K, 128 >> b);
      if (!ma) return -3;
      maps.a[m][b] = *ma;
    }
    a.rows_ptr[m] = rows_ptr[m]; a.act_out[m] = (bf16*)act_out[m];
  }
  a.N = N; a.K = K; a.scratch = scratch; a.scratch_rows = scratch_rows; a.arrived = arrived; a.reduced = reduced; a.fault = fault;
  return launch_ex(gateup_streamk_kernel, dim3(n_sms), dim3(kSkThreads), (size_t)kSkSmemBytes, s, pdl, maps, a) == cudaSuccess ? 0 : -3;
}
inline bool sk_gateup_init() {
  return cudaFuncSetAttribute(gateup_streamk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSkSmemBytes) == cudaSuccess;
}

}  // namespace tandem
