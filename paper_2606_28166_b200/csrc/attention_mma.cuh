// attention_mma.cuh - S5 over paged bf16 KV for the bf16 configs: split-KV GQA decode (S5a) and ragged catch-up /
// prefill attention (S5b) in one persistent kernel.
//
// Work unit = (attention item, kv head): the item's n_tok query tokens x G q-heads of the group form up to 64 rows
// (row = tok * G + g) that share every K/V byte of the unit's KV range [kv0, kv1).
//   producer warp : claims units (the first statically, the rest from an atomic counter, so no SM idles in the tail), looks
//                   pages up in the block table and streams them with TMA (cp.async.bulk.tensor, 128-byte swizzle, L2
//                   evict-first) into a ring of 64-token stages, each tagged with (unit, tile); it runs ahead across unit
//                   boundaries, so HBM never waits for a softmax.
//   4 consumer warps: S = Q K^T and O += P V on mma.sync.m16n8k16 (bf16 in, fp32 accumulate), online softmax in fp32
//                   registers. Rows <= 16 (decode, short catch-up): the warps split the pages of a stage and are merged at
//                   the end of the unit; more rows (long catch-up, prompt prefill): one 16-row m-tile per warp.
// The per-sequence q-tiles of a long run are dense contractions (q_len * G rows against the same KV) - the case SURVEY.md
// section 7 anticipates for tensor cores; for q_len = 1 the same tiles run at 25% MMA occupancy, which is still far
// above what HBM can feed. Q and P are rounded to bf16 (MMA inputs); scores, softmax state and O stay fp32.
// Output: attn_out (bf16) for unsplit items, else unnormalised partials (m, l, acc) combined by attn_combine_kernel.
#pragma once
#include "common.cuh"
#include "gemm_tcgen05.cuh"   // ptx:: mbarrier / TMA wrappers, TcGemmPlans (tensor-map encoder)

namespace tandem {

constexpr int kAmTileTok = 64;            // KV positions per ring stage = 4 pages
constexpr int kAmThreads = 160;           // 4 consumer warps + 1 producer warp
constexpr int kAmOPad = 8;                // floats of padding per scratch row (bank spread)

struct AttnMmaArgs {
  const int32_t* counts; const int32_t* item_row0; const int32_t* item_ntok; const int32_t* item_kv0; const int32_t* item_kv1;
  const int32_t* item_part; const int32_t* row_slot; const int32_t* row_pos; const int32_t* bt; int max_pages;
  const bf16* q;             // [rows, nq*D] bf16, RoPE applied
  bf16* out;                 // [rows, nq*D]
  float* part_acc;           // [parts, nq, D] unnormalised
  float2* part_ml;           // [parts, nq] (max of the scaled scores, sum)
  int nq, nkv; float scale;
  int row_base_k, row_base_v;  // tensor-map row of (page 0, kv head 0, token 0) of this layer's K / V pool
  int32_t* work_ctr;           // zeroed by the scheduler every step: units beyond the first gridDim.x are claimed dynamically
  int min_ntok;                // measurement only (bench.py, cfg 5): items with fewer query tokens are skipped; 0 = all items
};

namespace ptx {
__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ float ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
}  // namespace ptx

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

template <int D, int G, int STAGES>
__global__ void __launch_bounds__(kAmThreads, 2) paged_attention_mma_kernel(const __grid_constant__ Pair<CUtensorMap> maps, const __grid_constant__ Pair<AttnMmaArgs> ap) {
  constexpr int HALVES = D / 64;                    // 128-byte swizzle rows per K/V row
  constexpr int PAGE_BYTES = kPageTokens * D * 2;   // one (page, kv head) block of K or V
  constexpr int KV_BYTES = 4 * PAGE_BYTES;          // K (or V) part of a stage
  constexpr int STAGE_BYTES = 2 * KV_BYTES;
  constexpr int KS = D / 16;                        // k-steps of Q K^T
  constexpr int NT = D / 8;                         // n-tiles of O
  constexpr int OSTRIDE = D + kAmOPad;
  static_assert(D == 64 || D == 128, "head_dim");

  extern __shared__ uint8_t am_smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * STAGES];
  __shared__ float2 s_ml[4][16];
  __shared__ int2 s_meta[STAGES];                   // (unit, tile index) of the data in each stage; unit < 0: no more work

  pdl_trigger();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // units of both models share one index space (senior first) and one work counter: the tail is balanced across models
  const int nkv = ap.m[0].nkv;
  const int n_units0 = ap.m[0].counts[C_ITEMS] * nkv;   // written by the scheduler, complete long before this kernel can start
  const int n_units = n_units0 + ap.m[1].counts[C_ITEMS] * nkv;
  if ((int)blockIdx.x >= n_units) { pdl_wait(); return; }
  const uint32_t ring = (ptx::smem_u32(am_smem_raw) + 1023u) & ~1023u;
  float* scratch = reinterpret_cast<float*>(am_smem_raw + (ring - ptx::smem_u32(am_smem_raw)) + STAGES * STAGE_BYTES);   // [4][16][OSTRIDE]
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (uint32_t)(STAGES + s); };
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 4); }
    ptx::fence_mbar_init();
    ptx::prefetch_tmap(&maps.m[0]);
    ptx::prefetch_tmap(&maps.m[1]);
  }
  __syncthreads();
  pdl_wait();                                       // q and this step's K/V come from the predecessor (rope_append)

  if (warp == 4) {
    // ================================================================== producer
    const uint64_t pol = ptx::policy_evict_first();
    int it = 0;
    int u = blockIdx.x;
    while (true) {
      if (u < n_units) {
        const int mdl = u >= n_units0 ? 1 : 0;
        const AttnMmaArgs& a = ap.m[mdl];
        const CUtensorMap* tmap_kv = &maps.m[mdl];
        const int ul = u - mdl * n_units0;
        const int item = ul / nkv, kvh = ul - item * nkv;
        const int slot = a.row_slot[a.item_row0[item]];
        const int kv0 = a.item_kv0[item], kv1 = a.item_kv1[item];
        const int n_tiles = a.item_ntok[item] >= a.min_ntok ? (kv1 - kv0 + kAmTileTok - 1) / kAmTileTok : 0;   // a skipped item loads nothing: the consumers never see it
        const int32_t* btp = a.bt + (size_t)slot * a.max_pages + kv0 / kPageTokens;
        for (int ti = 0; ti < n_tiles; ++ti, ++it) {
          const int npg = min(4, (kv1 - kv0 - ti * kAmTileTok + kPageTokens - 1) / kPageTokens);
          const int pg = lane < npg ? btp[ti * 4 + lane] : 0;
          const int s = it % STAGES;
          if (lane == 0) {
            ptx::mbar_wait(empty_bar(s), (((uint32_t)(it / STAGES)) & 1u) ^ 1u);
            s_meta[s] = make_int2(u, ti);
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)(npg * 2 * PAGE_BYTES));
          }
          __syncwarp();
          if (lane < npg) {
            const int rk = a.row_base_k + (pg * a.nkv + kvh) * kPageTokens;
            const int rv = a.row_base_v + (pg * a.nkv + kvh) * kPageTokens;
            const uint32_t dk = ring + (uint32_t)(s * STAGE_BYTES + lane * PAGE_BYTES);
#pragma unroll
            for (int hh = 0; hh < HALVES; ++hh) {
              ptx::tma_load_2d(dk + hh * 2048, tmap_kv, hh * 64, rk, full_bar(s), pol);
              ptx::tma_load_2d(dk + KV_BYTES + hh * 2048, tmap_kv, hh * 64, rv, full_bar(s), pol);
            }
          }
        }
        int nu = 0;
        if (lane == 0) nu = atomicAdd(ap.m[0].work_ctr, 1) + (int)gridDim.x;
        u = __shfl_sync(0xffffffffu, nu, 0);
      } else {
        if (lane == 0) {   // sentinel stage: tells the consumers to stop
          const int s = it % STAGES;
          ptx::mbar_wait(empty_bar(s), (((uint32_t)(it / STAGES)) & 1u) ^ 1u);
          s_meta[s] = make_int2(-1, 0);
          ptx::mbar_arrive(full_bar(s));
        }
        break;
      }
    }
    return;
  }

  // ==================================================================== consumers
  const float c2 = ap.m[0].scale * 1.4426950408889634f;          // scores are kept as raw dots; p = 2^((s - m) * c2)
  const int quad = lane & 3, qrow = lane >> 2;
  // lane-constant parts of the ldmatrix addresses (see the layout notes in DESIGN.md section 6)
  const int kmat = lane >> 3;
  const int k_t = (lane & 7) + ((kmat >> 1) << 3);          // K: matrices (tok 0-7 | 8-15) x (chunk 2ks | 2ks+1)
  const int k_c = kmat & 1;
  const int v_t = (lane & 7) + ((kmat & 1) << 3);           // V (transposed): matrices (tok 0-7 | 8-15) x (chunk j | j+1)
  const int v_c = kmat >> 1;
  int it = 0;
  while (true) {
    ptx::mbar_wait(full_bar(it % STAGES), ((uint32_t)(it / STAGES)) & 1u);    // first stage of the next unit (or the sentinel)
    const int u = s_meta[it % STAGES].x;
    if (u < 0) break;
    const int mdl = u >= n_units0 ? 1 : 0;
    const AttnMmaArgs& a = ap.m[mdl];
    const int ul = u - mdl * n_units0;
    const int item = ul / nkv, kvh = ul - item * nkv;
    const int row0 = a.item_row0[item], n_tok = a.item_ntok[item], part = a.item_part[item];
    const int kv0 = a.item_kv0[item], kv1 = a.item_kv1[item];
    const int pos0 = a.row_pos[row0];
    const int n_rows = n_tok * G;
    const int m_tiles = (n_rows + 15) >> 4;
    const int mg = m_tiles == 1 ? 1 : (m_tiles == 2 ? 2 : 4);
    const int kvg = 4 / mg;
    const int mt = warp / kvg, kl = warp - mt * kvg;
    const bool active = mt < m_tiles;
    // the two rows of this lane in its m-tile
    const int gr0 = mt * 16 + qrow, gr1 = gr0 + 8;
    const int tk0 = gr0 / G, tk1 = gr1 / G;
    const int lim0 = gr0 < n_rows ? min(pos0 + tk0, kv1 - 1) : -1;   // last visible KV position of the row (-1: no row)
    const int lim1 = gr1 < n_rows ? min(pos0 + tk1, kv1 - 1) : -1;
    const int lim_max = __reduce_max_sync(0xffffffffu, max(lim0, lim1));
    const int lim_min = __reduce_min_sync(0xffffffffu, min(gr0 < n_rows ? lim0 : 0x7fffffff, gr1 < n_rows ? lim1 : 0x7fffffff));

    uint32_t qf[KS][4];
    {
      const bf16* q0 = a.q + ((size_t)(row0 + (gr0 < n_rows ? tk0 : 0)) * a.nq + kvh * G + (gr0 < n_rows ? gr0 - tk0 * G : 0)) * D;
      const bf16* q1 = a.q + ((size_t)(row0 + (gr1 < n_rows ? tk1 : 0)) * a.nq + kvh * G + (gr1 < n_rows ? gr1 - tk1 * G : 0)) * D;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        qf[ks][0] = *reinterpret_cast<const uint32_t*>(q0 + 16 * ks + 2 * quad);
        qf[ks][1] = *reinterpret_cast<const uint32_t*>(q1 + 16 * ks + 2 * quad);
        qf[ks][2] = *reinterpret_cast<const uint32_t*>(q0 + 16 * ks + 8 + 2 * quad);
        qf[ks][3] = *reinterpret_cast<const uint32_t*>(q1 + 16 * ks + 8 + 2 * quad);
      }
    }
    float o[NT][4];
#pragma unroll
    for (int j = 0; j < NT; ++j) { o[j][0] = 0.f; o[j][1] = 0.f; o[j][2] = 0.f; o[j][3] = 0.f; }
    float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;

    const int n_tiles = (kv1 - kv0 + kAmTileTok - 1) / kAmTileTok;
    for (int ti = 0; ti < n_tiles; ++ti, ++it) {
      const int s = it % STAGES;
      const int tile0 = kv0 + ti * kAmTileTok;
      const int npg = min(4, (kv1 - tile0 + kPageTokens - 1) / kPageTokens);
      if (ti > 0) ptx::mbar_wait(full_bar(s), ((uint32_t)(it / STAGES)) & 1u);
      if (active) {
        for (int p = kl; p < npg; p += kvg) {
          const int t0 = tile0 + p * kPageTokens;
          if (t0 > lim_max) break;                                   // wholly above the causal bound of this m-tile
          const uint32_t kp = ring + (uint32_t)(s * STAGE_BYTES + p * PAGE_BYTES), vp = kp + KV_BYTES;
          float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int ks = 0; ks < KS; ++ks) {
            const int ch = 2 * ks + k_c;
            uint32_t b0, b1, b2, b3;
            ptx::ldmatrix_x4(kp + (ch >> 3) * 2048 + k_t * 128 + (((ch & 7) ^ (k_t & 7)) << 4), b0, b1, b2, b3);
            ptx::mma_bf16_16816(s0, qf[ks], b0, b1);
            ptx::mma_bf16_16816(s1, qf[ks], b2, b3);
          }
          if (t0 + kPageTokens - 1 > lim_min) {                      // causal / range mask (warp-uniform test)
            const int c0 = t0 + 2 * quad;
            if (c0 > lim0) s0[0] = -INFINITY;  if (c0 + 1 > lim0) s0[1] = -INFINITY;
            if (c0 > lim1) s0[2] = -INFINITY;  if (c0 + 1 > lim1) s0[3] = -INFINITY;
            if (c0 + 8 > lim0) s1[0] = -INFINITY;  if (c0 + 9 > lim0) s1[1] = -INFINITY;
            if (c0 + 8 > lim1) s1[2] = -INFINITY;  if (c0 + 9 > lim1) s1[3] = -INFINITY;
          }
          float x0 = fmaxf(fmaxf(s0[0], s0[1]), fmaxf(s1[0], s1[1]));
          float x1 = fmaxf(fmaxf(s0[2], s0[3]), fmaxf(s1[2], s1[3]));
          x0 = fmaxf(x0, __shfl_xor_sync(0xffffffffu, x0, 1)); x0 = fmaxf(x0, __shfl_xor_sync(0xffffffffu, x0, 2));
          x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, 1)); x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, 2));
          const float n0 = fmaxf(m0, x0), n1 = fmaxf(m1, x1);
          const float u0 = n0 == -INFINITY ? 0.f : n0, u1 = n1 == -INFINITY ? 0.f : n1;   // no (-inf) - (-inf)
          const float al0 = ptx::ex2((m0 - u0) * c2), al1 = ptx::ex2((m1 - u1) * c2);
          m0 = n0; m1 = n1;
          const float p00 = ptx::ex2((s0[0] - u0) * c2), p01 = ptx::ex2((s0[1] - u0) * c2);
          const float p02 = ptx::ex2((s1[0] - u0) * c2), p03 = ptx::ex2((s1[1] - u0) * c2);
          const float p10 = ptx::ex2((s0[2] - u1) * c2), p11 = ptx::ex2((s0[3] - u1) * c2);
          const float p12 = ptx::ex2((s1[2] - u1) * c2), p13 = ptx::ex2((s1[3] - u1) * c2);
          l0 = l0 * al0 + (p00 + p01 + p02 + p03);
          l1 = l1 * al1 + (p10 + p11 + p12 + p13);
          uint32_t pa[4];
          pa[0] = pack_bf16x2(p00, p01); pa[1] = pack_bf16x2(p10, p11); pa[2] = pack_bf16x2(p02, p03); pa[3] = pack_bf16x2(p12, p13);
#pragma unroll
          for (int j = 0; j < NT; j += 2) {
            o[j][0] *= al0; o[j][1] *= al0; o[j][2] *= al1; o[j][3] *= al1;
            o[j + 1][0] *= al0; o[j + 1][1] *= al0; o[j + 1][2] *= al1; o[j + 1][3] *= al1;
            const int ch = j + v_c;
            uint32_t b0, b1, b2, b3;
            ptx::ldmatrix_x4_trans(vp + (ch >> 3) * 2048 + v_t * 128 + (((ch & 7) ^ (v_t & 7)) << 4), b0, b1, b2, b3);
            ptx::mma_bf16_16816(o[j], pa, b0, b1);
            ptx::mma_bf16_16816(o[j + 1], pa, b2, b3);
          }
        }
      }
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(empty_bar(s));
    }
    // ---- unit epilogue: per-warp state -> scratch, merge the kv-group warps of each m-tile, write out
    l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
    l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
    if (active) {
      float* sw = scratch + (size_t)warp * 16 * OSTRIDE;
      if (gr0 < n_rows) {
#pragma unroll
        for (int j = 0; j < NT; ++j) *reinterpret_cast<float2*>(sw + qrow * OSTRIDE + 8 * j + 2 * quad) = make_float2(o[j][0], o[j][1]);
        if (quad == 0) s_ml[warp][qrow] = make_float2(m0, l0);
      }
      if (gr1 < n_rows) {
#pragma unroll
        for (int j = 0; j < NT; ++j) *reinterpret_cast<float2*>(sw + (qrow + 8) * OSTRIDE + 8 * j + 2 * quad) = make_float2(o[j][2], o[j][3]);
        if (quad == 0) s_ml[warp][qrow + 8] = make_float2(m1, l1);
      }
    }
    ptx::bar_sync(1, 128);
    for (int idx = threadIdx.x; idx < n_rows * (D / 4); idx += 128) {
      const int gr = idx / (D / 4), d4 = idx - gr * (D / 4);
      const int mtile = gr >> 4, r = gr & 15;
      float M = -INFINITY;
      for (int k = 0; k < kvg; ++k) M = fmaxf(M, s_ml[mtile * kvg + k][r].x);
      const float Mu = M == -INFINITY ? 0.f : M;
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
      float L = 0.f;
      for (int k = 0; k < kvg; ++k) {
        const float2 ml = s_ml[mtile * kvg + k][r];
        const float w = ptx::ex2((ml.x - Mu) * c2);
        const float4 v = *reinterpret_cast<const float4*>(scratch + ((size_t)(mtile * kvg + k) * 16 + r) * OSTRIDE + 4 * d4);
        acc.x += w * v.x; acc.y += w * v.y; acc.z += w * v.z; acc.w += w * v.w;
        L += w * ml.y;
      }
      const int tok = gr / G, head = kvh * G + (gr - tok * G);
      if (part < 0) {
        const float inv = 1.f / L;
        uint2 pk;
        pk.x = pack_bf16x2(acc.x * inv, acc.y * inv); pk.y = pack_bf16x2(acc.z * inv, acc.w * inv);
        *reinterpret_cast<uint2*>(a.out + ((size_t)(row0 + tok) * a.nq + head) * D + 4 * d4) = pk;
      } else {
        *reinterpret_cast<float4*>(a.part_acc + ((size_t)(part + tok) * a.nq + head) * D + 4 * d4) = acc;
        if (d4 == 0) a.part_ml[(size_t)(part + tok) * a.nq + head] = make_float2(M * a.scale, L);
      }
    }
    ptx::bar_sync(1, 128);
  }
}

template <int D, int STAGES> constexpr int attn_mma_smem_bytes() {
  return 1024 + STAGES * 2 * 4 * kPageTokens * D * 2 + 4 * 16 * (D + kAmOPad) * 4;
}

}  // namespace tandem
