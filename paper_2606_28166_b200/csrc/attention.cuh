// attention.cuh - S5a split-KV GQA decode attention and S5b ragged catch-up attention over paged KV
// (DESIGN.md section 6). Plain ALUs (fp32 FMA), 128-bit loads of K/V, warp-shuffle reductions.
// One work unit = (attention item, kv head): all G = n_q/n_kv query heads of the group share every K/V load.
//   item = n_tok consecutive rows of one sequence x one KV range [kv0, kv1) (common.cuh StepTab): a single-q-tile
//   sequence is split along KV -> partial (m, l, acc) per row and split; q-tiles of longer runs are written directly.
// This kernel walks the rows of an item one by one on plain ALUs: it is the fp32 path (configs[0]) and the reference the
// tensor-core kernel of attention_mma.cuh is tested against.
// softmax(q.K^T / sqrt(d)) V with q-head a reading kv-head a / G (oracle/model.py states the same definition).
#pragma once
#include "common.cuh"

namespace tandem {

template <typename T> struct AttnArgs {
  const int32_t* counts; const int32_t* item_row0; const int32_t* item_ntok; const int32_t* item_kv0; const int32_t* item_kv1; const int32_t* item_part;
  const int32_t* row_slot; const int32_t* row_pos; const int32_t* bt; int max_pages;
  const float* q;            // [rows, nq*D] fp32, RoPE applied
  const T* kpool; const T* vpool;  // this layer: [pages, nkv, kPageTokens, D]
  T* out;                    // [rows, nq*D]
  float* part_acc;           // [parts, nq, D] unnormalised
  float2* part_ml;           // [parts, nq] (running max, sum)
  int nq, nkv; float scale;
};

template <typename T, int VEC> struct VecLoad;
template <> struct VecLoad<float, 4> {
  static __device__ __forceinline__ void ld(const float* p, float (&v)[4]) {
    const float4 t = *reinterpret_cast<const float4*>(p); v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
};
template <> struct VecLoad<bf16, 8> {
  static __device__ __forceinline__ void ld(const bf16* p, float (&v)[8]) {
    const uint4 t = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) { v[2 * i] = __uint_as_float(w[i] << 16); v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u); }
  }
};

constexpr int kAttnThreads = 128;
constexpr int kAttnTile = 64;   // KV positions per softmax tile

template <typename T, int D, int G>
__global__ void __launch_bounds__(kAttnThreads) paged_attention_kernel(const __grid_constant__ Pair<AttnArgs<T>> pp) {
  pdl_trigger(); pdl_wait();
  const AttnArgs<T>& a = pp.m[blockIdx.y];
  constexpr int VEC = 16 / (int)sizeof(T);
  constexpr int LPP = D / VEC;                   // lanes cooperating on one KV position
  constexpr int PPW = 32 / LPP;                  // positions per warp per iteration
  constexpr int NSG = (kAttnThreads / 32) * PPW; // sub-groups per CTA
  constexpr int ITER = kAttnTile / NSG;
  static_assert(LPP >= 1 && LPP <= 32 && (32 % LPP) == 0 && (kAttnTile % NSG) == 0, "unsupported head_dim");
  __shared__ float s_sc[G][kAttnTile];
  __shared__ float s_max[G];
  __shared__ int s_page[kAttnTile / kPageTokens];
  __shared__ float s_merge[kAttnThreads / 32][G][D];
  __shared__ float s_l[kAttnThreads / 32][G];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int sub = lane / LPP, ld_ = lane % LPP;   // sub-group within the warp, lane within the sub-group
  const int sg = warp * PPW + sub;
  const int n_units = a.counts[C_ITEMS] * a.nkv;

  for (int unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
    const int item = unit / a.nkv, kvh = unit - item * a.nkv;
    const int row0 = a.item_row0[item], n_tok = a.item_ntok[item], part0 = a.item_part[item];
    const int slot = a.row_slot[row0];
    const int kv0 = a.item_kv0[item];
    const int32_t* bt = a.bt + (size_t)slot * a.max_pages;
   for (int tok = 0; tok < n_tok; ++tok) {
    const int row = row0 + tok, part = part0 >= 0 ? part0 + tok : -1;
    const int kv1 = min(a.item_kv1[item], a.row_pos[row] + 1);   // causal bound of this row; may be <= kv0 (empty partial)

    float qv[G][VEC], acc[G][VEC], m_run[G], l_run[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
      const float* qp = a.q + (size_t)row * a.nq * D + (kvh * G + g) * D + ld_ * VEC;
#pragma unroll
      for (int e = 0; e < VEC; ++e) { qv[g][e] = qp[e] * a.scale; acc[g][e] = 0.f; }
      m_run[g] = -INFINITY; l_run[g] = 0.f;
    }

    for (int t0 = kv0; t0 < kv1; t0 += kAttnTile) {
      if (threadIdx.x < kAttnTile / kPageTokens) {
        const int pg = t0 / kPageTokens + threadIdx.x;   // t0 is a multiple of kAttnTile, hence of the page size
        s_page[threadIdx.x] = (pg * kPageTokens < kv1) ? bt[pg] : 0;
      }
      __syncthreads();
      // ---- phase 1: scores
      float kx[ITER][VEC];
#pragma unroll
      for (int i = 0; i < ITER; ++i) {
        const int pt = sg + i * NSG, pos = t0 + pt;
        if (pos < kv1) {
          const T* kp = a.kpool + (((size_t)s_page[pt / kPageTokens] * a.nkv + kvh) * kPageTokens + pt % kPageTokens) * D + ld_ * VEC;
          VecLoad<T, VEC>::ld(kp, kx[i]);
        } else {
#pragma unroll
          for (int e = 0; e < VEC; ++e) kx[i][e] = 0.f;
        }
      }
#pragma unroll
      for (int i = 0; i < ITER; ++i) {
        const int pt = sg + i * NSG, pos = t0 + pt;
#pragma unroll
        for (int g = 0; g < G; ++g) {
          float d = 0.f;
#pragma unroll
          for (int e = 0; e < VEC; ++e) d = fmaf(qv[g][e], kx[i][e], d);
#pragma unroll
          for (int o = LPP / 2; o > 0; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
          if (ld_ == 0) s_sc[g][pt] = pos < kv1 ? d : -INFINITY;
        }
      }
      __syncthreads();
      // ---- phase 2: tile max per head, rescale running state, probabilities in place
      for (int g = warp; g < G; g += kAttnThreads / 32) {
        const float mx = warp_max(fmaxf(s_sc[g][lane], s_sc[g][lane + 32]));
        if (lane == 0) s_max[g] = mx;
      }
      __syncthreads();
      float m_new[G];
#pragma unroll
      for (int g = 0; g < G; ++g) {
        m_new[g] = fmaxf(m_run[g], s_max[g]);
        const float alpha = __expf(m_run[g] - m_new[g]);   // exp(-inf) = 0 on the first tile
        l_run[g] *= alpha;
#pragma unroll
        for (int e = 0; e < VEC; ++e) acc[g][e] *= alpha;
      }
      for (int idx = threadIdx.x; idx < G * kAttnTile; idx += kAttnThreads) {
        const int g = idx / kAttnTile, pt = idx - g * kAttnTile;
        float mg = m_new[0];
#pragma unroll
        for (int gg = 1; gg < G; ++gg) mg = (g == gg) ? m_new[gg] : mg;
        s_sc[g][pt] = __expf(s_sc[g][pt] - mg);           // masked positions: exp(-inf) = 0
      }
#pragma unroll
      for (int g = 0; g < G; ++g) m_run[g] = m_new[g];
      __syncthreads();
      // ---- phase 3: acc += p V
#pragma unroll
      for (int i = 0; i < ITER; ++i) {
        const int pt = sg + i * NSG, pos = t0 + pt;
        if (pos < kv1) {
          const T* vp = a.vpool + (((size_t)s_page[pt / kPageTokens] * a.nkv + kvh) * kPageTokens + pt % kPageTokens) * D + ld_ * VEC;
          VecLoad<T, VEC>::ld(vp, kx[i]);
        } else {
#pragma unroll
          for (int e = 0; e < VEC; ++e) kx[i][e] = 0.f;
        }
      }
#pragma unroll
      for (int i = 0; i < ITER; ++i) {
        const int pt = sg + i * NSG;
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const float p = s_sc[g][pt];
          l_run[g] += p;
#pragma unroll
          for (int e = 0; e < VEC; ++e) acc[g][e] = fmaf(p, kx[i][e], acc[g][e]);
        }
      }
      __syncthreads();
    }

    // ---- merge the sub-groups (all share the same running max, so the merge is a plain sum)
#pragma unroll
    for (int g = 0; g < G; ++g) {
#pragma unroll
      for (int o = LPP; o < 32; o <<= 1) {
        l_run[g] += __shfl_xor_sync(0xffffffffu, l_run[g], o);
#pragma unroll
        for (int e = 0; e < VEC; ++e) acc[g][e] += __shfl_xor_sync(0xffffffffu, acc[g][e], o);
      }
      if (sub == 0) {
#pragma unroll
        for (int e = 0; e < VEC; ++e) s_merge[warp][g][ld_ * VEC + e] = acc[g][e];
        if (ld_ == 0) s_l[warp][g] = l_run[g];
      }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < G * D; idx += kAttnThreads) {
      const int g = idx / D, e = idx - g * D;
      float v = 0.f, l = 0.f;
#pragma unroll
      for (int w = 0; w < kAttnThreads / 32; ++w) { v += s_merge[w][g][e]; l += s_l[w][g]; }
      const int head = kvh * G + g;
      if (part < 0) {
        Elem<T>::st(a.out + (size_t)row * a.nq * D + head * D + e, v / l);
      } else {
        a.part_acc[((size_t)part * a.nq + head) * D + e] = v;
        if (e == 0) {
          float mg = m_run[0];
#pragma unroll
          for (int gg = 1; gg < G; ++gg) mg = (g == gg) ? m_run[gg] : mg;
          a.part_ml[(size_t)part * a.nq + head] = make_float2(mg, l);
        }
      }
    }
    __syncthreads();
   }
  }
}

// Combine the splits of a decode row: out = sum_i e^{m_i - m} acc_i / sum_i e^{m_i - m} l_i.
template <typename T> struct CombineArgs {
  const int32_t* counts; const int32_t* comb_row; const int32_t* comb_part0; const int32_t* comb_n; const int32_t* comb_stride;
  const int32_t* comb_gpart;   // optional extra partial per row (the row's part of a shared-prefix run), -1 = none
  const float* part_acc; const float2* part_ml; T* out; int nq, d;
};
// One warp per (row, head); lane = 4 consecutive dims; all partial loads of a row are independent (n <= kAttnMaxSplits).
template <typename T>
__global__ void __launch_bounds__(256) attn_combine_kernel(const __grid_constant__ Pair<CombineArgs<T>> pp) {
  pdl_trigger(); pdl_wait();
  const CombineArgs<T>& a = pp.m[blockIdx.y];
  const int n_units = a.counts[C_COMB] * a.nq;
  const int lane = threadIdx.x & 31;
  for (int unit = blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5); unit < n_units; unit += gridDim.x * (blockDim.x / 32)) {
    const int c = unit / a.nq, head = unit - c * a.nq;
    const int row = a.comb_row[c], p0 = a.comb_part0[c], n = a.comb_n[c], ps = a.comb_stride[c], gp = a.comb_gpart[c];
    // entry 0 = the shared-prefix partial (if any), entries 1.. = the row's own splits, in KV order
    float2 ml[kAttnMaxSplits + 1];
    int pi[kAttnMaxSplits + 1];
    float m = -INFINITY;
#pragma unroll
    for (int i = 0; i <= kAttnMaxSplits; ++i) {
      const bool on = i == 0 ? gp >= 0 : i - 1 < n;
      pi[i] = i == 0 ? gp : p0 + (i - 1) * ps;
      ml[i] = on ? a.part_ml[(size_t)pi[i] * a.nq + head] : make_float2(-INFINITY, 0.f);
      m = fmaxf(m, ml[i].x);
    }
    float l = 0.f, w[kAttnMaxSplits + 1];
#pragma unroll
    for (int i = 0; i <= kAttnMaxSplits; ++i) { w[i] = ml[i].x == -INFINITY ? 0.f : __expf(ml[i].x - m); l += w[i] * ml[i].y; }
    for (int e = 4 * lane; e < a.d; e += 128) {
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int i = 0; i <= kAttnMaxSplits; ++i) {
        if (i == 0 ? gp >= 0 : i - 1 < n) {
          const float4 t = ld4(a.part_acc + ((size_t)pi[i] * a.nq + head) * a.d + e);
          v.x += w[i] * t.x; v.y += w[i] * t.y; v.z += w[i] * t.z; v.w += w[i] * t.w;
        }
      }
      const float inv = 1.f / l;
      st4(a.out + (size_t)row * a.nq * a.d + head * a.d + e, make_float4(v.x * inv, v.y * inv, v.z * inv, v.w * inv));
    }
  }
}

}  // namespace tandem
