// attention_tcgen05.cuh - S5b for teacher-forced scoring (tandem_score): causal attention of whole
// prompt / stream chunks over the paged bf16 KV cache on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM).
//
// While scoring, every row of a step is a query and a sequence contributes hundreds of them: the q-tiles are dense contractions.
// The scheduler cuts each sequence's rows into q-tiles of 128 / G tokens (G = q-heads per kv-head), so that the (token, q-head of
// the group) pairs of a tile are the 128 rows of one UMMA M: row = tok * G + g, as in attention_mma.cuh. A work unit is
// (q-tile, kv head); the unit walks its causal KV range [0, pos0 + n_tok) in tiles of 128 positions (8 pages):
//   warp 0      : TMA - Q tile once per unit (3-D box: 64 dims x G heads x 128/G tokens per 128-byte-swizzled half), then the K and V
//                 pages of each KV tile, looked up in the block table, into single K and V buffers ([half][position][128 B]).
//   warp 1      : one elected thread issues S = Q K^T (both operands K-major in shared memory, N = 128) and O += P V with P read
//                 from TENSOR MEMORY (A operand in TMEM: the softmax warps overwrite S with bf16 P in place, so P never touches
//                 shared memory) and V as an MN-major shared-memory operand (V is stored position-major, the contraction runs over
//                 positions). MMAs execute in issue order, so S = Q K^T of the next tile is queued right behind O += P V.
//   warps 2-5   : one thread per row (TMEM lane quarter = warp % 4): row maximum, exp2, row sum, P packed to bf16 and stored back
//                 over S; the O accumulator is rescaled only when a row's maximum has grown by more than 2^8 since its reference
//                 (the rows keep their own reference; the final division by the row sum is exact either way).
// Two CTAs per SM (96 KB of shared memory, 256 TMEM columns each): while one CTA's rows are in the softmax, the other's MMAs
// keep the tensor pipe busy - the two q-tiles of a ping-pong schedule, arranged by the hardware scheduler instead of by hand.
// Units are claimed from an atomic counter, longest KV range first, the two models interleaved.
// Rounding points are those of attention_mma.cuh: q, k, v and P are bf16 (MMA inputs); scores, softmax state and O are fp32.
#pragma once
#include "attention_mma.cuh"

namespace tandem {

constexpr int kAtTileKv = 128;     // KV positions per tile = UMMA N of S = Q K^T
constexpr int kAtThreads = 192;
constexpr int kAtTmemCols = 256;   // S: columns [0, 128) (P as packed bf16 pairs over [0, 64)); O: columns [128, 128 + D)
constexpr int kAtHalfBytes = kAtTileKv * 128;   // one 64-dim half of a 128-row tile

namespace ptx {
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar, uint64_t policy) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
               ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(policy) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]: A is read from tensor memory (lane = row, two bf16 per 32-bit column)
__device__ __forceinline__ void umma_bf16_ta(uint32_t d_tmem, uint32_t a_tmem, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem), "r"(a_tmem), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
      : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
      ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
        "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]),
        "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]),
        "r"(v[30]), "r"(v[31])
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
}  // namespace ptx

// Shared-memory descriptor of an MN-major bf16 operand under the 128-byte swizzle: rows of the contraction dimension (KV positions)
// are 128 bytes = 64 elements of the MN dimension; 8 such rows form a 1024-byte swizzle atom (stride byte offset between atoms along
// the contraction); `lbo_bytes` separates the 64-element spans along MN (the two 64-dim halves of a head).
__device__ __forceinline__ uint64_t umma_desc_sw128_mn(uint32_t smem_addr, uint32_t lbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)(1024u >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

// barrier slots
enum { AT_Q_FULL = 0, AT_K_FULL, AT_V_FULL, AT_S_FULL, AT_P_READY, AT_PV_DONE, AT_NBARS };

template <int D>
__global__ void __launch_bounds__(kAtThreads, 2)
prefill_attention_tc_kernel(const __grid_constant__ Pair<CUtensorMap> kv_maps, const __grid_constant__ Pair<CUtensorMap> q_maps,
                            const __grid_constant__ Pair<AttnMmaArgs> ap, int G) {
  constexpr int HALVES = D / 64;
  constexpr int TILE_BYTES = HALVES * kAtHalfBytes;   // Q, K or V tile: [half][128 rows][128 B]
  constexpr int KS_QK = D / 16;                       // k-steps of S = Q K^T (contraction over head_dim)
  static_assert(D == 64 || D == 128, "head_dim");

  extern __shared__ uint8_t at_smem_raw[];
  __shared__ __align__(8) uint64_t bars[AT_NBARS];
  __shared__ uint32_t s_tmem;
  __shared__ int s_unit[2];

  pdl_trigger();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t base = (ptx::smem_u32(at_smem_raw) + 1023u) & ~1023u;
  const uint32_t q_s = base, k_s = base + TILE_BYTES, v_s = base + 2 * TILE_BYTES;
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto bar = [&](int i) { return bar0 + 8u * (uint32_t)i; };
  if (threadIdx.x == 0) {
    ptx::mbar_init(bar(AT_Q_FULL), 1); ptx::mbar_init(bar(AT_K_FULL), 1); ptx::mbar_init(bar(AT_V_FULL), 1);
    ptx::mbar_init(bar(AT_S_FULL), 1); ptx::mbar_init(bar(AT_P_READY), 128); ptx::mbar_init(bar(AT_PV_DONE), 1);
    ptx::fence_mbar_init();
    ptx::prefetch_tmap(&kv_maps.m[0]); ptx::prefetch_tmap(&kv_maps.m[1]);
    ptx::prefetch_tmap(&q_maps.m[0]); ptx::prefetch_tmap(&q_maps.m[1]);
  }
  if (warp == 1) ptx::tmem_alloc<kAtTmemCols>(ptx::smem_u32(&s_tmem));
  {  // a ragged last tile leaves pages of the V buffer untouched: they must hold finite values (P is exactly 0 there, 0 * NaN is not)
    uint8_t* z = at_smem_raw + (base - ptx::smem_u32(at_smem_raw));
    for (int i = threadIdx.x; i < 3 * TILE_BYTES / 16; i += kAtThreads) reinterpret_cast<uint4*>(z)[i] = make_uint4(0u, 0u, 0u, 0u);
    ptx::fence_proxy_async();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem = s_tmem;
  pdl_wait();                                       // q and this step's K/V come from the predecessor (rope_append)

  const int nkv = ap.m[0].nkv;
  const int n0 = ap.m[0].counts[C_ITEMS] * nkv, n1 = ap.m[1].counts[C_ITEMS] * nkv;
  const int n_units = n0 + n1, n_min = min(n0, n1);
  const float c2 = ap.m[0].scale * 1.4426950408889634f;
  const int tok_box = kAtTileKv / G;                // tokens per q-tile (the scheduler's tile_tok while scoring)
  uint32_t unit_it = 0, t_glob = 0;                 // units and KV tiles this CTA has been through: the barriers' phase parities
  int u = blockIdx.x;
  while (u < n_units) {
    int nxt = 0;
    if (threadIdx.x == 0) nxt = atomicAdd(ap.m[0].work_ctr, 1) + (int)gridDim.x;   // needed only at the end of this unit
    // claim order: the two models alternate while both have units, longest KV range (last q-tile) first
    int mdl, idx;
    if (u < 2 * n_min) { mdl = u & 1; idx = u >> 1; } else { mdl = n0 > n1 ? 0 : 1; idx = u - n_min; }
    const AttnMmaArgs& a = ap.m[mdl];
    const int item = a.counts[C_ITEMS] - 1 - idx / nkv, kvh = idx % nkv;
    const int row0 = a.item_row0[item], n_tok = a.item_ntok[item], kv1 = a.item_kv1[item];
    const int n_tiles = (kv1 + kAtTileKv - 1) / kAtTileKv;

    if (warp == 0) {
      // ================================================================== TMA producer
      const uint64_t pol_q = ptx::policy_evict_first(), pol_kv = ptx::policy_evict_last();   // K/V tiles are re-read by the other q-tiles of the sequence
      if (lane == 0) {
        ptx::mbar_expect_tx(bar(AT_Q_FULL), (uint32_t)(HALVES * tok_box * G * 128));
#pragma unroll
        for (int hh = 0; hh < HALVES; ++hh) ptx::tma_load_3d(q_s + hh * kAtHalfBytes, &q_maps.m[mdl], hh * 64, kvh * G, row0, bar(AT_Q_FULL), pol_q);
      }
      const int32_t* btp = a.bt + (size_t)a.row_slot[row0] * a.max_pages;
      const CUtensorMap* kvm = &kv_maps.m[mdl];
      for (int j = 0; j < n_tiles; ++j) {
        const uint32_t t = t_glob + (uint32_t)j;
        const int npg = min(8, (kv1 - j * kAtTileKv + kPageTokens - 1) / kPageTokens);
        const int pg = lane < npg ? btp[j * 8 + lane] : 0;
        const int prow = (pg * a.nkv + kvh) * kPageTokens;
        if (t > 0) ptx::mbar_wait(bar(AT_S_FULL), (t - 1) & 1u);      // K buffer free: S = Q K^T of the previous tile has completed
        if (lane == 0) ptx::mbar_expect_tx(bar(AT_K_FULL), (uint32_t)(npg * HALVES * 2048));
        __syncwarp();
        if (lane < npg) {
#pragma unroll
          for (int hh = 0; hh < HALVES; ++hh) ptx::tma_load_2d(k_s + hh * kAtHalfBytes + lane * 2048, kvm, hh * 64, a.row_base_k + prow, bar(AT_K_FULL), pol_kv);
        }
        if (t > 0) ptx::mbar_wait(bar(AT_PV_DONE), (t - 1) & 1u);     // V buffer free: O += P V of the previous tile has completed
        if (lane == 0) ptx::mbar_expect_tx(bar(AT_V_FULL), (uint32_t)(npg * HALVES * 2048));
        __syncwarp();
        if (lane < npg) {
#pragma unroll
          for (int hh = 0; hh < HALVES; ++hh) ptx::tma_load_2d(v_s + hh * kAtHalfBytes + lane * 2048, kvm, hh * 64, a.row_base_v + prow, bar(AT_V_FULL), pol_kv);
        }
      }
    } else if (warp == 1) {
      // ================================================================== MMA issue
      const uint32_t idesc_qk = umma_idesc_bf16(kAtTileKv);                 // M 128, N 128, both operands K-major
      const uint32_t idesc_pv = umma_idesc_bf16(D) | (1u << 16);            // M 128, N D, B (= V) MN-major
      const uint32_t tm_s = tmem, tm_o = tmem + 128u;
      auto issue_qk = [&]() {
        if (ptx::elect_one()) {
#pragma unroll
          for (int ks = 0; ks < KS_QK; ++ks) {
            const uint32_t off = (uint32_t)((ks >> 2) * kAtHalfBytes + (ks & 3) * 32);
            ptx::umma_bf16(tm_s, umma_desc_sw128(q_s + off), umma_desc_sw128(k_s + off), idesc_qk, ks > 0 ? 1u : 0u);
          }
          ptx::umma_commit(bar(AT_S_FULL));
        }
        __syncwarp();
      };
      ptx::mbar_wait(bar(AT_Q_FULL), unit_it & 1u);
      ptx::mbar_wait(bar(AT_K_FULL), t_glob & 1u);
      ptx::tc_fence_after();
      issue_qk();
      for (int j = 0; j < n_tiles; ++j) {
        const uint32_t t = t_glob + (uint32_t)j;
        const int n_ks = min(8, (kv1 - j * kAtTileKv + 15) >> 4);          // 16-position k-steps that hold visible positions
        ptx::mbar_wait(bar(AT_P_READY), t & 1u);
        ptx::mbar_wait(bar(AT_V_FULL), t & 1u);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          for (int ks = 0; ks < n_ks; ++ks)
            ptx::umma_bf16_ta(tm_o, tm_s + (uint32_t)(ks * 8), umma_desc_sw128_mn(v_s + ks * 2048, kAtHalfBytes), idesc_pv, (j > 0 || ks > 0) ? 1u : 0u);
          ptx::umma_commit(bar(AT_PV_DONE));
        }
        __syncwarp();
        if (j + 1 < n_tiles) {
          ptx::mbar_wait(bar(AT_K_FULL), (t + 1) & 1u);
          ptx::tc_fence_after();
          issue_qk();                                 // queued behind O += P V: MMAs execute in issue order, so S may alias P
        }
      }
    } else {
      // ================================================================== softmax, correction, epilogue: one thread per row
      const int quarter = warp & 3;
      const int row = quarter * 32 + lane;
      const uint32_t tm_row = tmem + ((uint32_t)(quarter * 32) << 16);
      const uint32_t tm_o = tm_row + 128u;
      const int tok = row / G, g = row - tok * G;
      const bool valid = row < n_tok * G;
      const int pos0 = a.row_pos[row0];
      const int lim = valid ? pos0 + tok : kv1 - 1;   // last visible KV position; rows beyond the tile compute on garbage and are not stored
      const int lim_min = __reduce_min_sync(0xffffffffu, lim);
      float m_ref = -INFINITY, l = 0.f;
      uint32_t v[32];
      for (int j = 0; j < n_tiles; ++j) {
        const uint32_t t = t_glob + (uint32_t)j;
        const int tile0 = j * kAtTileKv;
        const bool need_mask = tile0 + kAtTileKv - 1 > lim_min;    // warp-uniform
        ptx::mbar_wait(bar(AT_S_FULL), t & 1u);
        ptx::tc_fence_after();
        float mx = -INFINITY;
#pragma unroll 1
        for (int c = 0; c < 4; ++c) {
          ptx::tmem_ld32(tm_row + (uint32_t)(c * 32), v);
          ptx::tmem_ld_wait();
          if (need_mask) {
#pragma unroll
            for (int i = 0; i < 32; ++i) if (tile0 + c * 32 + i <= lim) mx = fmaxf(mx, __uint_as_float(v[i]));
          } else {
#pragma unroll
            for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(v[i]));
          }
        }
        if (j == 0) {
          m_ref = mx;                                 // position 0 is visible to every row: finite
        } else {
          const bool grow = (mx - m_ref) * c2 > 8.f;
          if (__any_sync(0xffffffffu, grow)) {        // rescale O and l to the new reference (a factor of 1 for rows that keep theirs)
            const float m2 = grow ? mx : m_ref;
            const float alpha = ptx::ex2((m_ref - m2) * c2);
            m_ref = m2; l *= alpha;
#pragma unroll 1
            for (int c = 0; c < D / 32; ++c) {
              ptx::tmem_ld32(tm_o + (uint32_t)(c * 32), v);
              ptx::tmem_ld_wait();
#pragma unroll
              for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * alpha);
              ptx::tmem_st32(tm_o + (uint32_t)(c * 32), v);
            }
          }
        }
        const float mb = m_ref * c2;
#pragma unroll 1
        for (int c = 0; c < 4; ++c) {
          ptx::tmem_ld32(tm_row + (uint32_t)(c * 32), v);
          ptx::tmem_ld_wait();
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            float p0 = ptx::ex2(fmaf(__uint_as_float(v[2 * i]), c2, -mb)), p1 = ptx::ex2(fmaf(__uint_as_float(v[2 * i + 1]), c2, -mb));
            if (need_mask) {
              if (tile0 + c * 32 + 2 * i > lim) p0 = 0.f;
              if (tile0 + c * 32 + 2 * i + 1 > lim) p1 = 0.f;
            }
            l += p0 + p1;
            pk[i] = pack_bf16x2(p0, p1);
          }
          ptx::tmem_st16(tm_row + (uint32_t)(c * 16), pk);   // P over S: columns [16c, 16c + 16) were consumed in this or an earlier chunk
        }
        ptx::tmem_st_wait();
        ptx::tc_fence_before();
        ptx::mbar_arrive(bar(AT_P_READY));
      }
      // ---- unit epilogue: O / l -> attn_out (bf16)
      ptx::mbar_wait(bar(AT_PV_DONE), (t_glob + (uint32_t)n_tiles - 1u) & 1u);
      ptx::tc_fence_after();
      const float inv = 1.f / l;
      bf16* orow = a.out + ((size_t)(row0 + (valid ? tok : 0)) * a.nq + kvh * G + (valid ? g : 0)) * D;
#pragma unroll 1
      for (int c = 0; c < D / 32; ++c) {
        ptx::tmem_ld32(tm_o + (uint32_t)(c * 32), v);
        ptx::tmem_ld_wait();
        if (valid) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            uint4 o4;
            o4.x = pack_bf16x2(__uint_as_float(v[8 * i]) * inv, __uint_as_float(v[8 * i + 1]) * inv);
            o4.y = pack_bf16x2(__uint_as_float(v[8 * i + 2]) * inv, __uint_as_float(v[8 * i + 3]) * inv);
            o4.z = pack_bf16x2(__uint_as_float(v[8 * i + 4]) * inv, __uint_as_float(v[8 * i + 5]) * inv);
            o4.w = pack_bf16x2(__uint_as_float(v[8 * i + 6]) * inv, __uint_as_float(v[8 * i + 7]) * inv);
            *reinterpret_cast<uint4*>(orow + c * 32 + 8 * i) = o4;
          }
        }
      }
      ptx::tc_fence_before();
    }
    // ---- unit boundary: every buffer (Q, K, V, S / P, O) is free again once all roles are through
    t_glob += (uint32_t)n_tiles;
    if (threadIdx.x == 0) s_unit[unit_it & 1u] = nxt;
    __syncthreads();
    ptx::tc_fence_after();
    u = s_unit[unit_it & 1u];
    ++unit_it;
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) ptx::tmem_dealloc<kAtTmemCols>(tmem);
}

template <int D> constexpr int attn_tc_smem_bytes() { return 1024 + 3 * (D / 64) * kAtHalfBytes; }

}  // namespace tandem
