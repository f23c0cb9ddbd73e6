// layer_tail.cuh - everything between two attention launches in ONE persistent kernel, for both models (bf16 configs):
//   LT_O     O projection of layer l                        (S6)   tcgen05 GEMM, split-K partials
//   LT_NORM1 residual add + RMSNorm(mlp_norm)                (S6)   element-wise
//   LT_GU    gate/up projection + SwiGLU epilogue            (S7)   tcgen05 GEMM
//   LT_DOWN  down projection                                 (S7)   tcgen05 GEMM, split-K partials
//   LT_NORM2 residual add + RMSNorm(attn_norm of l+1 | final) (S7/S2)
//   LT_QKV   QKV projection of layer l+1                     (S3)   tcgen05 GEMM, split-K partials
//   LT_ROPE  RoPE + KV append of layer l+1                   (S4)   element-wise
// One CTA per SM (grid = SM count, all resident). Phases are separated by grid barriers (one global counter per phase,
// zeroed by the scheduler), NOT by kernel boundaries, so the TMA producer warp never stops: weights do not depend on
// activations, and it streams the next phase's weight tiles into the shared-memory ring while the other warps finish the
// epilogue, wait at the barrier and run the element-wise phase. Only the activation boxes of a stage wait for the barrier.
// This removes the per-kernel fixed costs (launch, prologue, first TMA round trip, drain) that made the seven separate
// kernels take 190 us per layer for 62 us of weight streaming (profiles/launches_r1d.md).
//   warp 0    : weight TMA producer (never waits for a grid barrier: runs ahead as far as the ring allows)
//   warp 10   : activation TMA producer (same stage sequence, gated by the barrier of the producing phase)
//   warp 1    : MMA issuer (tcgen05.mma, one thread)
//   warps 2-9 : epilogue (tcgen05.ld -> global) and the element-wise phases
// GEMM units: (model, K-split, pair of adjacent 128-row weight tiles). The pair shares every activation tile (one 256-row
// TMA box of W, two M=128 accumulators in TMEM), which halves the activation traffic through the L2 fabric; units are
// dealt round-robin to the CTAs, and a trailing remainder of at most half a round is dealt as single tiles.
#pragma once
#include "gemm_tcgen05.cuh"

namespace tandem {

constexpr int kLtThreads = 352;             // weight-TMA warp, MMA warp, 8 epilogue / element-wise warps, activation-TMA warp
constexpr int kLtEpiThreads = 256;
constexpr int kLtMaxStages = 8;
constexpr int kLtRingBytes = 224 * 1024;     // 4 stages up to 192 token rows
constexpr int kLtSmemBytes = kLtRingBytes + 1024;
constexpr int kLtW2Bytes = 2 * kTcWBytes;          // a 256-row x 64 weight box

enum { LT_O = 0, LT_NORM1 = 1, LT_GU = 2, LT_DOWN = 3, LT_NORM2 = 4, LT_QKV = 5, LT_ROPE = 6, LT_NPHASE = 7 };

struct LtModel {
  const int32_t* counts;                // step table of this model (C_ROWS)
  float* x; float* gemm_out;            // residual stream [R,H]; split-K partials [S][row_cap][N]
  bf16* act; bf16* mlp_act; bf16* lm_in;
  const bf16* g_mlp; const bf16* g_next;  // gains of LT_NORM1 / LT_NORM2
  const int32_t* row_emit;              // last layer: LT_NORM2 writes only emitting rows, compacted, to lm_in; else null
  const int32_t* row_pos; const int32_t* row_kvslot;
  bf16* q; bf16* kpool; bf16* vpool;    // LT_ROPE targets (pools of layer l+1)
};
// Tensor maps live in device memory (written once by the host): weights [layer][gemm: 0 O, 1 gate/up, 2 down, 3 QKV][model]
// [box: 0 = 256 rows, 1 = 128 rows], activations [operand: 0 attn_out, 1 act, 2 mlp_act][model][box: 128, 64, 32, 16 rows].
// A thread issues a TMA box in ~0.1 us, so a 144-row activation tile goes out as 128 + 16 rows, not as nine 16-row boxes.
struct LtWMaps { CUtensorMap w[4][2][2]; };
struct LtAMaps { CUtensorMap a[3][2][4]; };
__device__ __forceinline__ int lt_gemm_idx(int p) { return p == LT_O ? 0 : (p == LT_GU ? 1 : (p == LT_DOWN ? 2 : 3)); }
__device__ __forceinline__ int lt_a_idx(int p) { return p == LT_O ? 0 : (p == LT_DOWN ? 2 : 1); }
struct LtArgs {
  LtModel m[2];
  int H, I, nq, nkv, d; float eps; const float2* rope_cs;
  int S_o, S_down, S_qkv, row_cap;
  int32_t* bar;                         // [LT_NPHASE] arrival counters of this launch
  int phase_mask;
  const LtWMaps* wm_l; const LtWMaps* wm_ln;   // weight maps of layer l (O, gate/up, down) and of layer l+1 (QKV)
  const LtAMaps* am;
  unsigned long long* dbg_ts;           // optional [2 + 2 * LT_NPHASE] globaltimer stamps written by CTA 0 (tuning aid), or null
};
__device__ __forceinline__ unsigned long long lt_now() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

struct LtGemm { int N, K, S, epi, dep; };   // dep: phase whose completion the activations wait for (-1: the previous kernel)
__device__ __forceinline__ LtGemm lt_gemm(const LtArgs& a, int p) {
  LtGemm g;
  if (p == LT_O) { g.N = a.H; g.K = a.nq * a.d; g.S = a.S_o; g.epi = kTcEpiPartial; g.dep = -1; }
  else if (p == LT_GU) { g.N = 2 * a.I; g.K = a.H; g.S = 1; g.epi = kTcEpiSwiGLU; g.dep = LT_NORM1; }
  else if (p == LT_DOWN) { g.N = a.H; g.K = a.I; g.S = a.S_down; g.epi = kTcEpiPartial; g.dep = LT_GU; }
  else { g.N = (a.nq + 2 * a.nkv) * a.d; g.K = a.H; g.S = a.S_qkv; g.epi = kTcEpiPartial; g.dep = (a.phase_mask >> LT_NORM2) & 1 ? LT_NORM2 : -1; }
  return g;
}
__device__ __forceinline__ bool lt_is_gemm(int p) { return p == LT_O || p == LT_GU || p == LT_DOWN || p == LT_QKV; }

// One accumulator fill: a unit (model, split, one or two weight tiles) x one chunk of <= 256 token rows.
struct LtUC { int phase, m, n0, ntile, kb0, kb1, r0, crow, split, N, epi; bool box256; };

// Walks the unit-chunks of this CTA in phase order. All roles run the same walker, so they agree on the sequence.
struct LtWalker {
  int p, v, chunk;
  __device__ __forceinline__ void start(int cta) { p = 0; v = cta; chunk = 0; }
  __device__ bool next(const LtArgs& a, int cta, int G, LtUC& o) {
    while (p < LT_NPHASE) {
      if (!lt_is_gemm(p) || !((a.phase_mask >> p) & 1)) { ++p; v = cta; chunk = 0; continue; }
      const LtGemm g = lt_gemm(a, p);
      const int T = (g.N + kTcTileN - 1) / kTcTileN, Tp = (T + 1) >> 1;
      const int n_dual = 2 * g.S * Tp;
      const int rem = n_dual % G;
      const int n_main = (n_dual > G && rem > 0 && 2 * rem <= G) ? n_dual - rem : n_dual;   // the remainder goes out as single tiles
      const int n_total = n_main + 2 * (n_dual - n_main);
      if (v >= n_total) { ++p; v = cta; chunk = 0; continue; }
      const bool dual = v < n_main;
      const int u = dual ? v : n_main + ((v - n_main) >> 1);
      const int pr = u % Tp, s = (u / Tp) % g.S, m = u / (Tp * g.S);
      const int tile = 2 * pr + (dual ? 0 : ((v - n_main) & 1));
      const int rows = a.m[m].counts[C_ROWS];
      const int n_chunks = (rows + kTcMaxRows - 1) / kTcMaxRows;
      if (tile >= T || chunk >= n_chunks) { v += G; chunk = 0; continue; }
      const int kb_total = (g.K + kTcBlockK - 1) / kTcBlockK;
      o.phase = p; o.m = m; o.n0 = tile * kTcTileN; o.ntile = dual ? min(2, T - tile) : 1; o.box256 = dual;
      o.kb0 = (int)((long long)kb_total * s / g.S); o.kb1 = (int)((long long)kb_total * (s + 1) / g.S);
      o.r0 = chunk * kTcMaxRows; o.crow = min(rows - o.r0, kTcMaxRows); o.split = s; o.N = g.N; o.epi = g.epi;
      ++chunk;
      return true;
    }
    return false;
  }
};

namespace ptx {
__device__ __forceinline__ int ld_acquire_gpu(const int32_t* p) { int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v; }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  return done != 0;
}
__device__ __forceinline__ void tmem_alloc_512(uint32_t smem_dst) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_dst) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_512(uint32_t taddr) { asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(taddr) : "memory"); }
}  // namespace ptx

// ---------------------------------------------------------------------------------------------- element-wise phases
// Executed by the 256 epilogue threads (tid 0..255) of every CTA; rows of both models are dealt round-robin to the CTAs.
// Data produced by other CTAs in this launch (split-K partials) is read with ld.global.cg: L1 is not coherent across SMs.
// Sum over one 128-thread row group (grp = 0 | 1, named barrier 2 + grp); red has 4 floats per group.
__device__ __forceinline__ float lt_group_sum(float v, float* red, int gt, int grp) {
  v = warp_sum(v);
  ptx::bar_sync(2 + grp, 128);
  if ((gt & 31) == 0) red[4 * grp + (gt >> 5)] = v;
  ptx::bar_sync(2 + grp, 128);
  return red[4 * grp] + red[4 * grp + 1] + red[4 * grp + 2] + red[4 * grp + 3];
}

// Two rows at a time per CTA (128 threads each): at ~1.7 rows per CTA per phase both are in flight together.
__device__ void lt_norm_phase(const LtArgs& a, int p, int cta, int G, int tid, float* red) {
  constexpr int VMAX = 16;                                  // float4 per thread: H <= 8192
  const int R0 = a.m[0].counts[C_ROWS], R1 = a.m[1].counts[C_ROWS];
  const int H = a.H, H4 = H >> 2;
  const int S = p == LT_NORM1 ? a.S_o : a.S_down;
  const size_t stride = (size_t)a.row_cap * H;
  const int grp = tid >> 7, gt = tid & 127;
  const int n_iter = (R0 + R1 + 2 * G - 1) / (2 * G);       // uniform trip count: the group barriers need every thread
  for (int itn = 0; itn < n_iter; ++itn) {
    const int g = (2 * itn + grp) * G + cta;
    const bool live = g < R0 + R1;
    const int m = (live && g >= R0) ? 1 : 0, r = live ? g - (m ? R0 : 0) : 0;
    const LtModel& M = a.m[m];
    float* xr = M.x + (size_t)r * H;
    const float* pr = M.gemm_out + (size_t)r * H;
    float4 v[VMAX];
#pragma unroll
    for (int i = 0; i < VMAX; ++i) {
      const int j4 = gt + i * 128;
      v[i] = (live && j4 < H4) ? ld4(xr + 4 * j4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (live) {
#pragma unroll 2
      for (int s = 0; s < S; ++s) {
#pragma unroll
        for (int i = 0; i < VMAX; ++i) {
          const int j4 = gt + i * 128;
          if (j4 < H4) v[i] = add4(v[i], __ldcg(reinterpret_cast<const float4*>(pr + s * stride + 4 * j4)));
        }
      }
    }
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < VMAX; ++i) {
      const int j4 = gt + i * 128;
      if (live && j4 < H4) st4(xr + 4 * j4, v[i]);
      ss += v[i].x * v[i].x + v[i].y * v[i].y + v[i].z * v[i].z + v[i].w * v[i].w;
    }
    const float inv = rsqrtf(lt_group_sum(ss, red, gt, grp) / (float)H + a.eps);
    int orow = r; bf16* dst = M.act; const bf16* gain = p == LT_NORM1 ? M.g_mlp : M.g_next;
    if (p == LT_NORM2 && M.row_emit) { orow = live ? M.row_emit[r] : -1; dst = M.lm_in; }
    if (!live || orow < 0) continue;
#pragma unroll
    for (int i = 0; i < VMAX; ++i) {
      const int j4 = gt + i * 128;
      if (j4 < H4) {
        const float4 gn = ld4(gain + 4 * j4);
        st4(dst + (size_t)orow * H + 4 * j4, make_float4(v[i].x * gn.x * inv, v[i].y * gn.y * inv, v[i].z * gn.z * inv, v[i].w * gn.w * inv));
      }
    }
  }
}

__device__ void lt_rope_phase(const LtArgs& a, int cta, int G, int tid) {
  const int R0 = a.m[0].counts[C_ROWS], R1 = a.m[1].counts[C_ROWS];
  const int nq = a.nq, nkv = a.nkv, d = a.d, half = d >> 1, hq = half >> 2;
  const int ld = (nq + 2 * nkv) * d, n_rot = (nq + nkv) * hq, n_v = nkv * (d >> 2);
  const int S = a.S_qkv;
  const size_t stride = (size_t)a.row_cap * ld;
  const int grp = tid >> 7, gt = tid & 127;
  for (int g = grp * G + cta; g < R0 + R1; g += 2 * G) {       // two rows at a time per CTA, 128 threads each
    const int m = g < R0 ? 0 : 1, r = g - (m ? R0 : 0);
    const LtModel& M = a.m[m];
    const int pos = M.row_pos[r], kvslot = M.row_kvslot[r];
    const int page = kvslot / kPageTokens, off = kvslot % kPageTokens;
    const float* src = M.gemm_out + (size_t)r * ld;
    for (int i = gt; i < n_rot + n_v; i += 128) {
      if (i < n_rot) {
        const int head = i / hq, j = (i - head * hq) << 2;
        float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f), x1 = x0;
#pragma unroll 4
        for (int s = 0; s < S; ++s) {
          x0 = add4(x0, __ldcg(reinterpret_cast<const float4*>(src + s * stride + head * d + j)));
          x1 = add4(x1, __ldcg(reinterpret_cast<const float4*>(src + s * stride + head * d + j + half)));
        }
        const float4 c01 = *reinterpret_cast<const float4*>(a.rope_cs + (size_t)pos * half + j);
        const float4 c23 = *reinterpret_cast<const float4*>(a.rope_cs + (size_t)pos * half + j + 2);
        const float4 ra = make_float4(x0.x * c01.x - x1.x * c01.y, x0.y * c01.z - x1.y * c01.w, x0.z * c23.x - x1.z * c23.y, x0.w * c23.z - x1.w * c23.w);
        const float4 rb = make_float4(x1.x * c01.x + x0.x * c01.y, x1.y * c01.z + x0.y * c01.w, x1.z * c23.x + x0.z * c23.y, x1.w * c23.z + x0.w * c23.w);
        if (head < nq) {
          st4(M.q + (size_t)r * nq * d + head * d + j, ra);
          st4(M.q + (size_t)r * nq * d + head * d + j + half, rb);
        } else {
          bf16* dst = M.kpool + (((size_t)page * nkv + (head - nq)) * kPageTokens + off) * d;
          st4(dst + j, ra); st4(dst + j + half, rb);
        }
      } else {
        const int e = (i - n_rot) << 2;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
        for (int s = 0; s < S; ++s) v = add4(v, __ldcg(reinterpret_cast<const float4*>(src + s * stride + (nq + nkv) * d + e)));
        const int kh = e / d;
        st4(M.vpool + (((size_t)page * nkv + kh) * kPageTokens + off) * d + (e - kh * d), v);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- the kernel
__global__ void __launch_bounds__(kLtThreads, 1) layer_tail_kernel(const __grid_constant__ LtArgs a) {
  extern __shared__ uint8_t lt_smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * kLtMaxStages + 2];
  __shared__ uint32_t tmem_base_smem;
  __shared__ float red[kLtEpiThreads / 32];

  pdl_trigger();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cta = blockIdx.x, G = gridDim.x;
  const int R0 = a.m[0].counts[C_ROWS], R1 = a.m[1].counts[C_ROWS];   // scheduler output: complete before this kernel can start
  if (R0 + R1 <= 0) { pdl_wait(); return; }                           // uniform over the grid
  const int nbox_max = (min(max(R0, R1), kTcMaxRows) + kTcRowBox - 1) / kTcRowBox;
  const int stage_bytes = kLtW2Bytes + nbox_max * kTcABoxBytes;
  const int n_stages = min(kLtMaxStages, kLtRingBytes / stage_bytes);

  const uint32_t ring = (ptx::smem_u32(lt_smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (uint32_t)(kLtMaxStages + s); };
  const uint32_t tmem_full_bar = bar0 + 8u * (2 * kLtMaxStages);
  const uint32_t tmem_empty_bar = tmem_full_bar + 8u;
  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { ptx::mbar_init(full_bar(s), 2); ptx::mbar_init(empty_bar(s), 1); }   // full: weight + activation producers
    ptx::mbar_init(tmem_full_bar, 1);
    ptx::mbar_init(tmem_empty_bar, 8);
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc_512(ptx::smem_u32(&tmem_base_smem));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  if (warp == 0) {
    // ===== weight producer: runs ahead of the activations across phase boundaries, bounded only by free ring slots.
    // (One thread issues a TMA box in ~0.1-0.2 us, so weights and activations are issued by different warps.)
    {
      const uint64_t pol_w = ptx::policy_evict_first();
      LtWalker ww; ww.start(cta);
      LtUC uw;
      int nw = 0;
      while (ww.next(a, cta, G, uw)) {
        const int gi = lt_gemm_idx(uw.phase);
        const CUtensorMap* mw = &(gi == 3 ? a.wm_ln : a.wm_l)->w[gi][uw.m][uw.box256 ? 0 : 1];
        for (int kb = uw.kb0; kb < uw.kb1; ++kb, ++nw) {
          const int s = nw % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(nw / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)(uw.box256 ? kLtW2Bytes : kTcWBytes));
            ptx::tma_load_2d(ring + (uint32_t)(s * stage_bytes), mw, kb * kTcBlockK, uw.n0, full_bar(s), pol_w);
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 10) {
    // ===== activation producer: same stage sequence, gated by the grid barrier of the phase that produces the operand
    {
      const uint64_t pol_a = ptx::policy_evict_last();
      LtWalker wa; wa.start(cta);
      LtUC ua;
      int na = 0;
      uint32_t passed = 0; bool prev_kernel_done = false;
      while (wa.next(a, cta, G, ua)) {
        const int dep = lt_gemm(a, ua.phase).dep;
        if (dep < 0) { if (!prev_kernel_done) { pdl_wait(); prev_kernel_done = true; } }
        else if (!((passed >> dep) & 1u)) {
          while (ptx::ld_acquire_gpu(a.bar + dep) < G) { }
          passed |= 1u << dep;
          ptx::fence_proxy_async();
        }
        const int nbox = (ua.crow + kTcRowBox - 1) / kTcRowBox;
        const CUtensorMap* ma = a.am->a[lt_a_idx(ua.phase)][ua.m];
        for (int kb = ua.kb0; kb < ua.kb1; ++kb, ++na) {
          const int s = na % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(na / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            ptx::mbar_expect_tx(full_bar(s), (uint32_t)(nbox * kTcABoxBytes));
            const uint32_t dst = ring + (uint32_t)(s * stage_bytes) + kLtW2Bytes;
            int j = 0;                                     // rows issued so far, in 16-row units: greedy 128 / 64 / 32 / 16-row boxes
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              const int bx = 8 >> b;
              while (nbox - j >= bx) { ptx::tma_load_2d(dst + j * kTcABoxBytes, ma + b, kb * kTcBlockK, ua.r0 + j * kTcRowBox, full_bar(s), pol_a); j += bx; }
            }
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (all lanes run the loop, one elected lane issues: see ptx::elect_one)
    {
      LtWalker w; w.start(cta);
      LtUC u;
      int it = 0, acc_it = 0;
      long long dbg_full = 0, dbg_empty = 0;
      while (w.next(a, cta, G, u)) {
        const int ncols = ((u.crow + kTcRowBox - 1) / kTcRowBox) * kTcRowBox;
        const uint32_t idesc = umma_idesc_bf16(ncols);
        long long t0 = clock64();
        ptx::mbar_wait(tmem_empty_bar, ((uint32_t)acc_it & 1u) ^ 1u);
        dbg_empty += clock64() - t0;
        ptx::tc_fence_after();
        for (int kb = u.kb0; kb < u.kb1; ++kb, ++it) {
          const int s = it % n_stages;
          t0 = clock64();
          ptx::mbar_wait(full_bar(s), (uint32_t)(it / n_stages) & 1u);
          dbg_full += clock64() - t0;
          if (a.dbg_ts && cta == 0 && lane == 0 && u.phase == LT_GU && kb - u.kb0 < 8 && acc_it < 2) a.dbg_ts[20 + (kb - u.kb0)] = lt_now();
          ptx::tc_fence_after();
          const uint32_t sw = ring + (uint32_t)(s * stage_bytes);
          const uint64_t da = umma_desc_sw128(sw + kLtW2Bytes);
          if (ptx::elect_one()) {
            for (int j = 0; j < u.ntile; ++j) {
              const uint64_t dw = umma_desc_sw128(sw + j * kTcWBytes);
#pragma unroll
              for (int k = 0; k < kTcBlockK / 16; ++k)
                ptx::umma_bf16(tmem_base + (uint32_t)(j * kTcMaxRows), dw + (uint64_t)(2 * k), da + (uint64_t)(2 * k), idesc, (kb > u.kb0 || k > 0) ? 1u : 0u);
            }
            ptx::umma_commit(empty_bar(s));
          }
          __syncwarp();
        }
        if (ptx::elect_one()) ptx::umma_commit(tmem_full_bar);
        __syncwarp();
        ++acc_it;
      }
      if (a.dbg_ts && cta == 0 && lane == 0) { a.dbg_ts[16] = (unsigned long long)dbg_full; a.dbg_ts[17] = (unsigned long long)dbg_empty; a.dbg_ts[18] = (unsigned long long)it; a.dbg_ts[19] = (unsigned long long)n_stages; }
    }
  } else {
    // ===== epilogue warps (TMEM quarter q = warp % 4) + element-wise phases
    const int q = warp & 3;
    const int grp = (warp - 2) >> 2;          // two warps per TMEM quarter: group 0 takes tile 0 (or the even column chunks), group 1 the rest
    const int tid = threadIdx.x - 64;
    if (a.dbg_ts && cta == 0 && tid == 0) a.dbg_ts[0] = lt_now();
    pdl_wait();   // before the first global write: the previous kernel may still read q / KV / attn_out
    if (a.dbg_ts && cta == 0 && tid == 0) a.dbg_ts[1] = lt_now();
    LtWalker w; w.start(cta);
    LtUC u;
    bool have = w.next(a, cta, G, u);
    int acc_it = 0;
    auto phase_arrive = [&](int p) {
      __threadfence();
      ptx::bar_sync(1, kLtEpiThreads);
      if (tid == 0) atomicAdd(a.bar + p, 1);
    };
    auto phase_wait = [&](int p) {
      if (tid == 0) { while (ptx::ld_acquire_gpu(a.bar + p) < G) { } }
      ptx::bar_sync(1, kLtEpiThreads);
    };
    for (int p = 0; p < LT_NPHASE; ++p) {
      if (!((a.phase_mask >> p) & 1)) continue;
      if (lt_is_gemm(p)) {
        while (have && u.phase == p) {
          const LtModel& M = a.m[u.m];
          ptx::mbar_wait(tmem_full_bar, (uint32_t)acc_it & 1u);
          ptx::tc_fence_after();
          for (int j = 0; j < u.ntile; ++j) {
            if (u.ntile == 2 && j != grp) continue;
            const int n = u.n0 + j * kTcTileN + q * 32 + lane;
            for (int c0 = (u.ntile == 2 ? 0 : 32 * grp); c0 < u.crow; c0 += (u.ntile == 2 ? 32 : 64)) {
              uint32_t v[32];
              ptx::tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(j * kTcMaxRows + c0), v);
              ptx::tmem_ld_wait();
              if (u.epi == kTcEpiPartial) {
                float* outp = M.gemm_out + (size_t)u.split * ((size_t)a.row_cap * u.N);
                if (n < u.N) {
#pragma unroll
                  for (int k = 0; k < 32; ++k)
                    if (c0 + k < u.crow) outp[(size_t)(u.r0 + c0 + k) * u.N + n] = __uint_as_float(v[k]);
                }
              } else {   // rows interleaved gate/up: see gemm_tcgen05_kernel
                const bool odd = lane & 1;
                const int i = n >> 1, I = u.N >> 1;
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                  const float mine = __uint_as_float(odd ? v[16 + k] : v[k]);
                  const float send = __uint_as_float(odd ? v[k] : v[16 + k]);
                  const float recv = __shfl_xor_sync(0xffffffffu, send, 1);
                  const float gate = odd ? recv : mine, up = odd ? mine : recv;
                  const int r = c0 + (odd ? 16 : 0) + k;
                  if (r < u.crow && n < u.N) M.mlp_act[(size_t)(u.r0 + r) * I + i] = __float2bfloat16_rn(gate / (1.f + expf(-gate)) * up);
                }
              }
            }
          }
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(tmem_empty_bar);
          ++acc_it;
          have = w.next(a, cta, G, u);
        }
        phase_arrive(p);
        if (a.dbg_ts && cta == 0 && tid == 0) a.dbg_ts[2 + 2 * p + 1] = lt_now();
      } else {
        const int dep = p == LT_NORM1 ? LT_O : (p == LT_NORM2 ? LT_DOWN : LT_QKV);
        if ((a.phase_mask >> dep) & 1) phase_wait(dep);
        if (a.dbg_ts && cta == 0 && tid == 0) a.dbg_ts[2 + 2 * p] = lt_now();
        if (p == LT_ROPE) lt_rope_phase(a, cta, G, tid);
        else lt_norm_phase(a, p, cta, G, tid, red);
        phase_arrive(p);
        if (a.dbg_ts && cta == 0 && tid == 0) a.dbg_ts[2 + 2 * p + 1] = lt_now();
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc_512(tmem_base);
}

}  // namespace tandem
