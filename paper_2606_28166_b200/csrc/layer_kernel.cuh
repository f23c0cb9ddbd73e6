// layer_kernel.cuh - everything between two attention launches in ONE persistent kernel, for both models (bf16 configs):
//   O projection (S6) -> residual + RMSNorm -> gate/up projection + SwiGLU (S7) -> down projection -> residual + RMSNorm (S7/S2)
//   -> QKV projection of the next layer (S3) -> RoPE + KV append (S4)
// as a list of phases (LkPhase) executed by one CTA per SM. Why one kernel: at ~128 token rows per model the four projections
// of a layer stream 402 MB of weights (62 us at HBM speed) but took 129 us as four launches plus 36 us in four element-wise
// launches - every launch pays its prologue, first TMA round trip, epilogue and drain, and one-tile-per-CTA grids leave a
// partial last wave (gate/up: 304 tiles on 296 slots). Here
//   * the weight-TMA warp never stops: weights depend on nothing, so it streams the next phase's tiles into the ring while the
//     other warps finish an epilogue, wait at a grid barrier or run an element-wise phase;
//   * GEMM work is cut stream-K style: the (weight tile, k-block) units of a projection are dealt as CONTIGUOUS, EQUAL ranges,
//     so every SM streams the same number of weight bytes whatever the tile count; a tile cut by a range boundary is completed
//     from fp32 partial planes (summed in k order by the consumer phase: deterministic) or, for gate/up whose SwiGLU epilogue
//     needs the whole sum, by the CTA that owns the tile's first k-block, which adds the later pieces' partials (they were
//     computed at the START of their owners' ranges, so it does not wait in practice);
//   * a unit is a PAIR of adjacent 128-row weight tiles sharing every activation stage (two M = 128 accumulators), which halves
//     the activation bytes an SM pulls from L2 per weight byte (the ingest limit of the one-tile kernel, profiles/gemm_sweep_r1.md);
//   * accumulators are double-buffered in TMEM (2 x 2 x 128 columns at <= 128 token rows), so the tcgen05.ld epilogue of a
//     piece overlaps the MMAs of the next.
// Partition (a function of the shapes and the SM count only, so the summation order of every output element is independent of
// the batch): each model's units are cut into NR = SMs / 2 ranges. Both models active: CTA c serves model c / NR, range c % NR,
// with tile pairs. One model active (solo decoding, the first prefill): its range r is served by CTAs r and r + NR, one 128-row
// half of every pair each - the same k-ranges, hence bit-identical sums - so all SMs stream.
//   warp 0: weight TMA   warp 10: activation TMA (gated by the barrier of the producing phase)   warp 1: MMA issuer
//   warps 2-9: epilogue (tcgen05.ld -> global) and the element-wise phases
#pragma once
#include "gemm_tcgen05.cuh"

namespace tandem {

constexpr int kLkThreads = 352;
constexpr int kLkEpiThreads = 256;
constexpr int kLkMaxStages = 8;
constexpr int kLkRingBytes = 224 * 1024;
constexpr int kLkSmemBytes = kLkRingBytes + 1024;
constexpr int kLkMaxPhases = 8;
constexpr int kLkPairRows = 2 * kTcTileN;                 // weight rows of a tile pair
constexpr long long kLkSpinLimit = 4000000000ll;          // ~2 s of SM clocks: a wait this long means a lost signal - give up, flag, do not hang the GPU

enum { LK_GEMM_PARTIAL = 0, LK_GEMM_SWIGLU = 1, LK_NORM = 2, LK_ROPE = 3 };
enum { LK_A_ATTN = 0, LK_A_ACT = 1, LK_A_MLP = 2 };       // activation operands: attn_out, act, mlp_act

struct LkPhase {
  int type;
  int N, K;        // GEMM: out features, in features
  int wmap;        // GEMM: index into the weight tensor-map table (entry = [model][box: 256 | 128 rows])
  int amap;        // GEMM: LK_A_*
  int dep;         // GEMM: phase whose completion the activations wait for (-1: the previous kernel)
  int src;         // NORM / ROPE: the GEMM phase whose partial planes it sums
  int last;        // NORM: 1 = the final norm: only emitting rows, written compactly to lm_in
};

struct LkModel {
  const int32_t* counts;
  float* x; float* gemm_out;              // residual stream [R, H]; fp32 partial planes [plane][row_cap][N] (and the gate/up fix-up scratch)
  bf16* act; bf16* mlp_act; bf16* lm_in;
  const bf16* gain[kLkMaxPhases];         // NORM phases: the RMSNorm gain
  const int32_t* row_emit; const int32_t* row_pos; const int32_t* row_kvslot;
  bf16* q; bf16* kpool; bf16* vpool;      // ROPE targets
};

struct LkArgs {
  LkModel m[2];
  LkPhase ph[kLkMaxPhases]; int n_phases;
  int H, nq, nkv, d; float eps; const float2* rope_cs; int row_cap;
  int32_t* bar;                  // [kLkMaxPhases] arrival counters of this launch (zeroed by the scheduler every step)
  int32_t* flag;                 // [2 models][2 halves][NR] gate/up fix-up flags of this launch (zeroed by the scheduler)
  int32_t* abort_flag;           // set when a wait timed out (results invalid); sticky until tandem_reset
  const CUtensorMap* wmaps;      // device table [wmap][model][2]
  const CUtensorMap* amaps;      // device table [LK_A_*][model][4: 128, 64, 32, 16-row boxes]
  int dbg_flags;                 // timing experiments only (tandem_test_gemm_time): bit 0 = skip the activation loads (results are garbage)
  unsigned long long* dbg_ts;    // optional (tandem_test_set_option "layer_debug"): 32 globaltimer stamps / cycle counts per CTA, else null
};
__device__ __forceinline__ unsigned long long lk_now() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

// ---------------------------------------------------------------------------------------------- partition arithmetic (host and device)
// Two regimes. DT <= NR (the narrow projections: QKV, O, down): a 2-D split - S = NR / DT k-slices per tile pair, range
// r = t * S + j holds k-blocks [j KB / S, (j + 1) KB / S) of pair t: one piece per CTA, S planes per pair. DT > NR (gate/up): stream-K -
// the DT * KB units in tile-major order cut into NR contiguous, equal ranges (a range may end one pair and begin the next).
struct LkGeo { int DT, KB, NRp, S; long long U; };
__host__ __device__ __forceinline__ LkGeo lk_geo(int N, int K, int NR) {
  LkGeo g;
  g.DT = (N + kLkPairRows - 1) / kLkPairRows; g.KB = (K + kTcBlockK - 1) / kTcBlockK;
  g.U = (long long)g.DT * g.KB;
  if (g.DT <= NR) { g.S = NR / g.DT; if (g.S > g.KB) g.S = g.KB; g.NRp = g.S * g.DT; }     // every slice holds at least one k-block
  else { g.S = 0; g.NRp = NR; }
  return g;
}
__host__ __device__ __forceinline__ long long lk_range_begin(const LkGeo& g, int r) {
  if (g.S) { const int t = r / g.S, j = r - t * g.S; return (long long)t * g.KB + (long long)j * g.KB / g.S; }
  return g.U * r / g.NRp;
}
__host__ __device__ __forceinline__ int lk_range_of(const LkGeo& g, long long x) {      // the range that holds unit x
  if (g.S) { const int t = (int)(x / g.KB), kk = (int)(x - (long long)t * g.KB); return t * g.S + ((kk + 1) * g.S + g.KB - 1) / g.KB - 1; }
  return (int)(((x + 1) * g.NRp + g.U - 1) / g.U) - 1;
}
// partial planes of tile pair t = ranges that intersect it; plane index of range r = r - first
__host__ __device__ __forceinline__ int lk_first_range(const LkGeo& g, int t) { return lk_range_of(g, (long long)t * g.KB); }
__host__ __device__ __forceinline__ int lk_plane_count(const LkGeo& g, int t) {
  return lk_range_of(g, (long long)(t + 1) * g.KB - 1) - lk_first_range(g, t) + 1;
}
inline int lk_max_planes(int N, int K, int NR) {
  const LkGeo g = lk_geo(N, K, NR);
  int mx = 1;
  for (int t = 0; t < g.DT; ++t) mx = std::max(mx, lk_plane_count(g, t));
  return mx;
}

namespace ptx {
__device__ __forceinline__ int ld_acquire_gpu(const int32_t* p) { int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v; }
__device__ __forceinline__ void st_release_gpu(int32_t* p, int v) { asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc_512(uint32_t smem_dst) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_dst) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_512(uint32_t taddr) { asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(taddr) : "memory"); }
}  // namespace ptx

// Bounded spin on a global counter / flag written by other CTAs of this launch (all CTAs are co-resident: grid <= SM count).
__device__ __forceinline__ void lk_spin_ge(const int32_t* p, int target, int32_t* abort_flag) {
  const long long t0 = clock64();
  int it = 0;
  while (ptx::ld_acquire_gpu(p) < target) {
    if ((++it & 1023) == 0 && (clock64() - t0 > kLkSpinLimit || ptx::ld_acquire_gpu(abort_flag) != 0)) { atomicExch(abort_flag, 1); break; }
  }
}

// This CTA's place in the partition.
struct LkCta {
  int m;        // model it serves
  int r;        // range index (compared with each phase's NRp)
  int half;     // solo mode: which 128-row half of every tile pair
  int pair;     // 1 = tile pairs (both models active), 0 = single tiles (one model active)
  int rows;     // token rows of that model this step
  bool idle;    // no GEMM work at all (odd SM count, or solo mode beyond 2 NR)
};
__device__ __forceinline__ LkCta lk_cta(int cta, int G, int R0, int R1) {
  LkCta c;
  const int NR = G / 2;
  c.r = cta % NR;
  if (R0 > 0 && R1 > 0) { c.pair = 1; c.m = cta / NR; c.half = 0; c.idle = cta >= 2 * NR; if (c.idle) c.m = 0; }
  else { c.pair = 0; c.m = R0 > 0 ? 0 : 1; c.half = cta / NR; c.idle = cta >= 2 * NR; }
  c.rows = c.m == 0 ? R0 : R1;
  return c;
}

// One accumulator fill: (phase, tile pair or single tile, k-range, chunk of <= 256 token rows).
struct LkPiece {
  int phase, type, N;
  int t, n0, ntile;        // tile pair index, first weight row, weight tiles (1 | 2)
  int k0, k1;              // k-block range
  int r0, crow;            // token-row chunk
  int plane;               // PARTIAL: plane this piece writes
  int final_;              // SWIGLU: 1 = holds the tile's first k-block: runs the epilogue (after adding ranges wait_lo..wait_hi)
  int wait_lo, wait_hi;    // SWIGLU final piece: later ranges whose partials it adds (empty if wait_lo > wait_hi)
  int last_chunk;          // this is the last row chunk of the (tile, k-range)
};

// Walks this CTA's pieces in phase order. Every warp role runs its own copy, so all agree on the sequence.
struct LkWalker {
  const LkArgs* a; LkCta c; int NR;
  int p; bool init; long long u, uend; int chunk; LkGeo g;
  __device__ __forceinline__ void start(const LkArgs* a_, const LkCta& c_, int G) { a = a_; c = c_; NR = G / 2; p = 0; init = false; chunk = 0; u = uend = 0; }
  __device__ bool next(LkPiece& o) {
    while (p < a->n_phases) {
      const LkPhase& ph = a->ph[p];
      if (ph.type > LK_GEMM_SWIGLU || c.idle) { ++p; init = false; continue; }
      if (!init) {
        g = lk_geo(ph.N, ph.K, NR);
        if (c.r >= g.NRp) { ++p; continue; }
        u = lk_range_begin(g, c.r); uend = lk_range_begin(g, c.r + 1); chunk = 0; init = true;
      }
      if (u >= uend) { ++p; init = false; continue; }
      const int t = (int)(u / g.KB), k0 = (int)(u - (long long)t * g.KB);
      const int k1 = (int)min((long long)g.KB, k0 + (uend - u));
      const int n0 = t * kLkPairRows + c.half * kTcTileN;
      const int n_chunks = (c.rows + kTcMaxRows - 1) / kTcMaxRows;
      if (n0 >= ph.N) { u += k1 - k0; continue; }            // solo mode, second half of a last odd tile: nothing there
      o.phase = p; o.type = ph.type; o.N = ph.N; o.t = t; o.n0 = n0;
      o.ntile = c.pair ? ((n0 + kTcTileN < ph.N) ? 2 : 1) : 1;
      o.k0 = k0; o.k1 = k1;
      o.r0 = chunk * kTcMaxRows; o.crow = min(c.rows - o.r0, kTcMaxRows);
      const int first = lk_first_range(g, t);
      o.plane = c.r - first;
      o.final_ = k0 == 0;
      o.wait_lo = c.r + 1; o.wait_hi = k1 < g.KB ? lk_range_of(g, (long long)(t + 1) * g.KB - 1) : c.r;
      o.last_chunk = chunk == n_chunks - 1;
      if (++chunk == n_chunks) { chunk = 0; u += k1 - k0; }
      return true;
    }
    return false;
  }
};

// ---------------------------------------------------------------------------------------------- element-wise phases
// Executed by the 256 epilogue threads (tid 0..255) of every CTA; rows of both models are dealt round-robin to the CTAs, two
// rows at a time per CTA (128 threads each). Partial planes written by other CTAs of this launch are read with ld.global.cg
// (L1 is not coherent across SMs); a column block of 256 outputs has lk_plane_count planes, summed in k order.
__device__ __forceinline__ float lk_group_sum(float v, float* red, int gt, int grp) {
  v = warp_sum(v);
  ptx::bar_sync(2 + grp, 128);
  if ((gt & 31) == 0) red[4 * grp + (gt >> 5)] = v;
  ptx::bar_sync(2 + grp, 128);
  return red[4 * grp] + red[4 * grp + 1] + red[4 * grp + 2] + red[4 * grp + 3];
}

constexpr int kLkMaxPairs = 1024;    // tile pairs per projection (N <= 262,144) - the plane-count table in shared memory

// Plane counts of every tile pair of GEMM phase `src`, once per phase into shared memory (lk_plane_count costs 64-bit divisions).
__device__ __forceinline__ void lk_fill_plane_counts(const LkPhase& src, int NR, int tid, uint8_t* cnt_tab) {
  const LkGeo g = lk_geo(src.N, src.K, NR);
  for (int t = tid; t < g.DT && t < kLkMaxPairs; t += kLkEpiThreads) cnt_tab[t] = (uint8_t)lk_plane_count(g, t);
  ptx::bar_sync(1, kLkEpiThreads);
}
__device__ __forceinline__ float4 lk_zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }

// x[r,:] += sum of the partial planes (k order); act = RMSNorm(x; gain). Planes are read four at a time for all of the thread's
// column groups (20 independent 16-byte loads in flight at H = 2560): the phase is two L2 round trips, not one per plane.
template <int VMAX>                                         // float4 per thread (128 threads per row): H <= 512 VMAX
__device__ void lk_norm_phase(const LkArgs& a, int p, int cta, int G, int tid, float* red, const uint8_t* cnt_tab) {
  const int R0 = a.m[0].counts[C_ROWS], R1 = a.m[1].counts[C_ROWS];
  const int H = a.H, H4 = H >> 2;
  const size_t stride = (size_t)a.row_cap * H;
  const int grp = tid >> 7, gt = tid & 127;
  int cnt[VMAX], maxc = 0;
#pragma unroll
  for (int i = 0; i < VMAX; ++i) {
    const int j4 = gt + i * 128;
    cnt[i] = j4 < H4 ? cnt_tab[(4 * j4) / kLkPairRows] : 0;
    maxc = max(maxc, cnt[i]);
  }
  const int n_iter = (R0 + R1 + 2 * G - 1) / (2 * G);       // uniform trip count: the group barriers need every thread
  for (int itn = 0; itn < n_iter; ++itn) {
    const int gi = (2 * itn + grp) * G + cta;
    const bool live = gi < R0 + R1;
    const int m = (live && gi >= R0) ? 1 : 0, r = live ? gi - (m ? R0 : 0) : 0;
    const LkModel& M = a.m[m];
    float* xr = M.x + (size_t)r * H;
    const float* pr = M.gemm_out + (size_t)r * H + 4 * gt;
    const bf16* gain = M.gain[p];
    float4 v[VMAX], gn[VMAX];
#pragma unroll
    for (int i = 0; i < VMAX; ++i) {
      const int j4 = gt + i * 128;
      const bool on = live && j4 < H4;
      v[i] = on ? ld4(xr + 4 * j4) : lk_zero4();
      gn[i] = on ? ld4(gain + 4 * j4) : lk_zero4();
    }
    if (live) {
      for (int s0 = 0; s0 < maxc; s0 += 4) {
        float4 q[4][VMAX];
#pragma unroll
        for (int ss = 0; ss < 4; ++ss) {
#pragma unroll
          for (int i = 0; i < VMAX; ++i) {
            q[ss][i] = lk_zero4();
            if (s0 + ss < cnt[i]) q[ss][i] = __ldcg(reinterpret_cast<const float4*>(pr + (size_t)(s0 + ss) * stride + 512 * i));
          }
        }
#pragma unroll
        for (int ss = 0; ss < 4; ++ss) {
#pragma unroll
          for (int i = 0; i < VMAX; ++i) v[i] = add4(v[i], q[ss][i]);     // an absent plane adds +0: exact
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
    const float inv = rsqrtf(lk_group_sum(ss, red, gt, grp) / (float)H + a.eps);
    int orow = r; bf16* dst = M.act;
    if (a.ph[p].last) { orow = live ? M.row_emit[r] : -1; dst = M.lm_in; }
    if (!live || orow < 0) continue;
#pragma unroll
    for (int i = 0; i < VMAX; ++i) {
      const int j4 = gt + i * 128;
      if (j4 < H4) st4(dst + (size_t)orow * H + 4 * j4, make_float4(v[i].x * gn[i].x * inv, v[i].y * gn[i].y * inv, v[i].z * gn[i].z * inv, v[i].w * gn[i].w * inv));
    }
  }
}

// q, k, v of a row = sums of the QKV partial planes; RoPE on q and k (pairs (j, j + d/2), table built in double at init); q -> bf16
// buffer, k / v -> the model's pages. An item is a PAIR of float4 column groups: a rotation pair (c, c + d/2) of a q or k head, or two
// groups of v. A thread takes four items at a time and reads two planes of all eight groups per round trip.
__device__ void lk_rope_phase(const LkArgs& a, int p, int cta, int G, int tid, const uint8_t* cnt_tab) {
  const int R0 = a.m[0].counts[C_ROWS], R1 = a.m[1].counts[C_ROWS];
  const int nq = a.nq, nkv = a.nkv, d = a.d, half = d >> 1, hq = half >> 2;
  const int ld = (nq + 2 * nkv) * d, n_rot = (nq + nkv) * hq, n_vp = nkv * (d >> 3), vbase = (nq + nkv) * d;
  const int n_items = n_rot + n_vp;
  const size_t stride = (size_t)a.row_cap * ld;
  const int grp = tid >> 7, gt = tid & 127;
  for (int gi = grp * G + cta; gi < R0 + R1; gi += 2 * G) {       // two rows at a time per CTA, 128 threads each
    const int m = gi < R0 ? 0 : 1, r = gi - (m ? R0 : 0);
    const LkModel& M = a.m[m];
    const int pos = M.row_pos[r], kvslot = M.row_kvslot[r];
    const int page = kvslot / kPageTokens, off = kvslot % kPageTokens;
    const float* srcp = M.gemm_out + (size_t)r * ld;
    for (int i0 = gt; i0 < n_items; i0 += 4 * 128) {
      int c0[4], c1[4], cn0[4], cn1[4], maxc = 0;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int i = i0 + b * 128;
        if (i < n_rot) { const int head = i / hq; c0[b] = head * d + ((i - head * hq) << 2); c1[b] = c0[b] + half; }
        else { c0[b] = vbase + ((i - n_rot) << 2); c1[b] = c0[b] + (n_vp << 2); }
        const bool on = i < n_items;
        if (!on) { c0[b] = 0; c1[b] = 0; }
        cn0[b] = on ? cnt_tab[c0[b] / kLkPairRows] : 0; cn1[b] = on ? cnt_tab[c1[b] / kLkPairRows] : 0;
        maxc = max(maxc, max(cn0[b], cn1[b]));
      }
      float4 x0[4], x1[4];
#pragma unroll
      for (int b = 0; b < 4; ++b) { x0[b] = lk_zero4(); x1[b] = lk_zero4(); }
      for (int s0 = 0; s0 < maxc; s0 += 2) {
        float4 q0[2][4], q1[2][4];
#pragma unroll
        for (int ss = 0; ss < 2; ++ss) {
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            q0[ss][b] = lk_zero4(); q1[ss][b] = lk_zero4();
            if (s0 + ss < cn0[b]) q0[ss][b] = __ldcg(reinterpret_cast<const float4*>(srcp + (size_t)(s0 + ss) * stride + c0[b]));
            if (s0 + ss < cn1[b]) q1[ss][b] = __ldcg(reinterpret_cast<const float4*>(srcp + (size_t)(s0 + ss) * stride + c1[b]));
          }
        }
#pragma unroll
        for (int ss = 0; ss < 2; ++ss) {
#pragma unroll
          for (int b = 0; b < 4; ++b) { x0[b] = add4(x0[b], q0[ss][b]); x1[b] = add4(x1[b], q1[ss][b]); }
        }
      }
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int i = i0 + b * 128;
        if (i >= n_items) continue;
        if (i < n_rot) {
          const int head = i / hq, j = (i - head * hq) << 2;
          const float4 c01 = *reinterpret_cast<const float4*>(a.rope_cs + (size_t)pos * half + j);       // (cos, sin) of pairs j, j+1
          const float4 c23 = *reinterpret_cast<const float4*>(a.rope_cs + (size_t)pos * half + j + 2);
          const float4 u0 = x0[b], u1 = x1[b];
          const float4 ra = make_float4(u0.x * c01.x - u1.x * c01.y, u0.y * c01.z - u1.y * c01.w, u0.z * c23.x - u1.z * c23.y, u0.w * c23.z - u1.w * c23.w);
          const float4 rb = make_float4(u1.x * c01.x + u0.x * c01.y, u1.y * c01.z + u0.y * c01.w, u1.z * c23.x + u0.z * c23.y, u1.w * c23.z + u0.w * c23.w);
          if (head < nq) {
            st4(M.q + (size_t)r * nq * d + head * d + j, ra);
            st4(M.q + (size_t)r * nq * d + head * d + j + half, rb);
          } else {
            bf16* dst = M.kpool + (((size_t)page * nkv + (head - nq)) * kPageTokens + off) * d;
            st4(dst + j, ra); st4(dst + j + half, rb);
          }
        } else {
          const int e0 = (i - n_rot) << 2, e1 = e0 + (n_vp << 2);
          const int kh0 = e0 / d, kh1 = e1 / d;
          st4(M.vpool + (((size_t)page * nkv + kh0) * kPageTokens + off) * d + (e0 - kh0 * d), x0[b]);
          st4(M.vpool + (((size_t)page * nkv + kh1) * kPageTokens + off) * d + (e1 - kh1 * d), x1[b]);
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- the kernel
__global__ void __launch_bounds__(kLkThreads, 1) layer_kernel(const __grid_constant__ LkArgs a) {
  extern __shared__ uint8_t lk_smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * kLkMaxStages + 4];
  __shared__ uint32_t tmem_base_smem;
  __shared__ float red[kLkEpiThreads / 32];
  __shared__ uint8_t cnt_tab[kLkMaxPairs];

  pdl_trigger();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cta = blockIdx.x, G = gridDim.x;
  const int R0 = a.m[0].counts[C_ROWS], R1 = a.m[1].counts[C_ROWS];   // scheduler output: complete before this kernel can start
  if (R0 + R1 <= 0) { pdl_wait(); return; }                           // uniform over the grid
  const LkCta c = lk_cta(cta, G, R0, R1);
  unsigned long long* const dts = a.dbg_ts ? a.dbg_ts + (size_t)cta * 32 : nullptr;   // this CTA's 32 debug words
  unsigned long long* const trace = (a.dbg_ts && (cta == 0 || cta == G - 1)) ? a.dbg_ts + (size_t)G * 32 + (cta ? 192 : 0) : nullptr;   // [3][64]: issue, full, commit of the SwiGLU phase's stages
  const int wbytes = c.pair ? 2 * kTcWBytes : kTcWBytes;
  const int ncols_max = ((min(c.rows, kTcMaxRows) + kTcRowBox - 1) / kTcRowBox) * kTcRowBox;
  const int stage_bytes = wbytes + (ncols_max / kTcRowBox) * kTcABoxBytes;
  const int n_stages = min(kLkMaxStages, kLkRingBytes / stage_bytes);
  // accumulators: a piece needs ntile * ncols columns; two buffers of 256 columns when that fits, else one of 512
  const int nbuf = ((c.pair ? 2 : 1) * ncols_max <= 256) ? 2 : 1;
  const uint32_t tile_cols = (c.pair && ncols_max > 128) ? 256u : 128u;

  const uint32_t ring = (ptx::smem_u32(lk_smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (uint32_t)(kLkMaxStages + s); };
  auto tmem_full_bar = [&](int b) { return bar0 + 8u * (uint32_t)(2 * kLkMaxStages + b); };
  auto tmem_empty_bar = [&](int b) { return bar0 + 8u * (uint32_t)(2 * kLkMaxStages + 2 + b); };
  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { ptx::mbar_init(full_bar(s), 2); ptx::mbar_init(empty_bar(s), 1); }   // full: weight + activation producers
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(tmem_full_bar(b), 1); ptx::mbar_init(tmem_empty_bar(b), 8); }
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc_512(ptx::smem_u32(&tmem_base_smem));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  if (warp == 0) {
    // ===== weight producer: runs ahead of the activations across phase boundaries, bounded only by free ring slots
    const uint64_t pol_w = ptx::policy_evict_first();
    LkWalker w; w.start(&a, c, G);
    LkPiece pc;
    int n = 0, ntr = 0;
    while (w.next(pc)) {
      const CUtensorMap* mw = a.wmaps + ((size_t)(a.ph[pc.phase].wmap * 2 + c.m) * 2 + (c.pair ? 0 : 1));
      for (int kb = pc.k0; kb < pc.k1; ++kb, ++n) {
        const int s = n % n_stages;
        ptx::mbar_wait(empty_bar(s), ((uint32_t)(n / n_stages) & 1u) ^ 1u);
        if (trace && pc.type == LK_GEMM_SWIGLU && ntr < 64 && lane == 0) trace[ntr++] = lk_now();
        if (ptx::elect_one()) {
          ptx::mbar_expect_tx(full_bar(s), (uint32_t)wbytes);
          if (a.dbg_flags & 2) ptx::tma_load_2d(ring + (uint32_t)(s * stage_bytes), mw, 0, (pc.t * ((a.ph[pc.phase].K + kTcBlockK - 1) / kTcBlockK) + kb) * kLkPairRows + c.half * kTcTileN, full_bar(s), pol_w);
          else
          ptx::tma_load_2d(ring + (uint32_t)(s * stage_bytes), mw, kb * kTcBlockK, pc.n0, full_bar(s), pol_w);
        }
        __syncwarp();
      }
    }
  } else if (warp == 10) {
    // ===== activation producer: same stage sequence, gated by the grid barrier of the phase that produces the operand
    const uint64_t pol_a = ptx::policy_evict_last();
    LkWalker w; w.start(&a, c, G);
    LkPiece pc;
    int n = 0;
    uint32_t passed = 0; bool prev_kernel_done = false;
    while (w.next(pc)) {
      const int dep = a.ph[pc.phase].dep;
      if (dep < 0) { if (!prev_kernel_done) { pdl_wait(); prev_kernel_done = true; } }
      else if (!((passed >> dep) & 1u)) {
        lk_spin_ge(a.bar + dep, G, a.abort_flag);
        passed |= 1u << dep;
        ptx::fence_proxy_async();                            // other SMs' generic-proxy stores, acquired above, before this warp's TMA reads
      }
      const int nbox = (pc.crow + kTcRowBox - 1) / kTcRowBox;
      const CUtensorMap* ma = a.amaps + (size_t)(a.ph[pc.phase].amap * 2 + c.m) * 4;
      for (int kb = pc.k0; kb < pc.k1; ++kb, ++n) {
        const int s = n % n_stages;
        ptx::mbar_wait(empty_bar(s), ((uint32_t)(n / n_stages) & 1u) ^ 1u);
        if (ptx::elect_one()) {
          if (a.dbg_flags & 1) { ptx::mbar_arrive(full_bar(s)); } else {
          ptx::mbar_expect_tx(full_bar(s), (uint32_t)(nbox * kTcABoxBytes));
          const uint32_t dst = ring + (uint32_t)(s * stage_bytes) + (uint32_t)wbytes;
          int j = 0;                                         // rows issued so far, in 16-row units: greedy 128 / 64 / 32 / 16-row boxes
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const int bx = 8 >> b;
            while (nbox - j >= bx) { ptx::tma_load_2d(dst + j * kTcABoxBytes, ma + b, kb * kTcBlockK, pc.r0 + j * kTcRowBox, full_bar(s), pol_a); j += bx; }
          }
          }
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (all lanes run the loop, one elected lane issues: see ptx::elect_one)
    LkWalker w; w.start(&a, c, G);
    LkPiece pc;
    int n = 0, i = 0;
    long long dbg_full = 0, dbg_empty = 0;
    const bool dbg = dts != nullptr;
    int dbg_phase = -1, ntr = 0;
    while (w.next(pc)) {
      const int buf = nbuf == 2 ? (i & 1) : 0, use = nbuf == 2 ? (i >> 1) : i;
      const int ncols = ((pc.crow + kTcRowBox - 1) / kTcRowBox) * kTcRowBox;
      const uint32_t idesc = umma_idesc_bf16(ncols);
      long long t0 = dbg ? clock64() : 0;
      ptx::mbar_wait(tmem_empty_bar(buf), ((uint32_t)use & 1u) ^ 1u);
      if (dbg) dbg_empty += clock64() - t0;
      ptx::tc_fence_after();
      const uint32_t acc = tmem_base + (uint32_t)buf * 256u;
      for (int kb = pc.k0; kb < pc.k1; ++kb, ++n) {
        const int s = n % n_stages;
        if (dbg) t0 = clock64();
        ptx::mbar_wait(full_bar(s), (uint32_t)(n / n_stages) & 1u);
        if (dbg) { dbg_full += clock64() - t0; if (pc.phase != dbg_phase) { dbg_phase = pc.phase; if (lane == 0) dts[16 + pc.phase] = lk_now(); } }
        if (trace && pc.type == LK_GEMM_SWIGLU && ntr < 64 && lane == 0) trace[64 + ntr] = lk_now();
        ptx::tc_fence_after();
        const uint32_t sw = ring + (uint32_t)(s * stage_bytes);
        const uint64_t da = umma_desc_sw128(sw + (uint32_t)wbytes);
        if (ptx::elect_one()) {
          for (int j = 0; j < pc.ntile; ++j) {
            const uint64_t dw = umma_desc_sw128(sw + (uint32_t)(j * kTcWBytes));
#pragma unroll
            for (int k = 0; k < kTcBlockK / 16; ++k)
              ptx::umma_bf16(acc + (uint32_t)j * tile_cols, dw + (uint64_t)(2 * k), da + (uint64_t)(2 * k), idesc, (kb > pc.k0 || k > 0) ? 1u : 0u);
          }
          ptx::umma_commit(empty_bar(s));
        }
        __syncwarp();
        if (trace && pc.type == LK_GEMM_SWIGLU && ntr < 64 && lane == 0) { trace[128 + ntr] = lk_now(); ++ntr; }
      }
      if (ptx::elect_one()) ptx::umma_commit(tmem_full_bar(buf));
      __syncwarp();
      ++i;
    }
    if (dbg && lane == 0) { dts[24] = (unsigned long long)dbg_full; dts[25] = (unsigned long long)dbg_empty; dts[26] = (unsigned long long)n; dts[27] = (unsigned long long)(n_stages * 1000 + nbuf); }
  } else {
    // ===== epilogue warps (TMEM lane quarter q = warp % 4) + element-wise phases
    const int q = warp & 3;
    const int grp = (warp - 2) >> 2;          // two warps per TMEM quarter: group g takes tile g of a pair (single tile: alternate 32-column chunks)
    const int tid = threadIdx.x - 64;
    const bool dbg = dts && tid == 0;
    if (dbg) dts[0] = lk_now();
    pdl_wait();   // before the first global write: the previous kernel may still read q / KV / attn_out
    if (dbg) dts[1] = lk_now();
    LkWalker w; w.start(&a, c, G);
    LkPiece pc;
    bool have = w.next(pc);
    int i = 0;
    auto phase_arrive = [&](int p) {
      __threadfence();
      ptx::bar_sync(1, kLkEpiThreads);
      if (tid == 0) atomicAdd(a.bar + p, 1);
    };
    auto phase_wait = [&](int p) {
      if (tid == 0) lk_spin_ge(a.bar + p, G, a.abort_flag);
      ptx::bar_sync(1, kLkEpiThreads);
    };
    for (int p = 0; p < a.n_phases; ++p) {
      const int type = a.ph[p].type;
      if (type <= LK_GEMM_SWIGLU) {
        if (dbg) dts[2 + 2 * p] = lk_now();
        while (have && pc.phase == p) {
          const LkModel& M = a.m[c.m];
          const int buf = nbuf == 2 ? (i & 1) : 0, use = nbuf == 2 ? (i >> 1) : i;
          const uint32_t acc = tmem_base + (uint32_t)buf * 256u;
          ptx::mbar_wait(tmem_full_bar(buf), (uint32_t)use & 1u);
          ptx::tc_fence_after();
          const bool swiglu = type == LK_GEMM_SWIGLU;
          const int n_add = (swiglu && pc.final_) ? pc.wait_hi - pc.wait_lo + 1 : 0;
          if (n_add > 0) {   // the later pieces of this tile were computed at the start of their owners' ranges
            if (tid == 0) for (int rr = pc.wait_lo; rr <= pc.wait_hi; ++rr) lk_spin_ge(a.flag + (c.m * 2 + c.half) * (G / 2) + rr, 1, a.abort_flag);
            ptx::bar_sync(1, kLkEpiThreads);
          }
          for (int j = 0; j < pc.ntile; ++j) {
            if (pc.ntile == 2 && j != grp) continue;
            const int nl = (c.pair ? j : c.half) * kTcTileN + q * 32 + lane;     // column within the tile pair
            const int n = pc.t * kLkPairRows + nl;
            for (int c0 = (pc.ntile == 2 ? 0 : 32 * grp); c0 < pc.crow; c0 += (pc.ntile == 2 ? 32 : 64)) {
              uint32_t v[32];
              ptx::tmem_ld32(acc + ((uint32_t)(q * 32) << 16) + (uint32_t)j * tile_cols + (uint32_t)c0, v);
              ptx::tmem_ld_wait();
              if (!swiglu) {
                float* outp = M.gemm_out + (size_t)pc.plane * ((size_t)a.row_cap * pc.N);
                if (n < pc.N) {
#pragma unroll
                  for (int k = 0; k < 32; ++k)
                    if (c0 + k < pc.crow) outp[(size_t)(pc.r0 + c0 + k) * pc.N + n] = __uint_as_float(v[k]);
                }
              } else if (!pc.final_) {   // raw partial sums into this range's scratch slot [range][row][256]
                float* sp = M.gemm_out + ((size_t)c.r * a.row_cap + pc.r0 + c0) * kLkPairRows + nl;
#pragma unroll
                for (int k = 0; k < 32; ++k)
                  if (c0 + k < pc.crow) sp[(size_t)k * kLkPairRows] = __uint_as_float(v[k]);
              } else {
                for (int rr = pc.wait_lo; rr <= pc.wait_lo + n_add - 1; ++rr) {       // ascending k order
                  const float* sp = M.gemm_out + ((size_t)rr * a.row_cap + pc.r0 + c0) * kLkPairRows + nl;
#pragma unroll
                  for (int k = 0; k < 32; ++k)
                    if (c0 + k < pc.crow) v[k] = __float_as_uint(__uint_as_float(v[k]) + __ldcg(sp + (size_t)k * kLkPairRows));
                }
                // rows interleaved gate/up (2i = gate_i, 2i+1 = up_i): even lane finishes columns [0,16), odd lane [16,32)
                const bool odd = lane & 1;
                const int ii = n >> 1, I = pc.N >> 1;
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                  const float mine = __uint_as_float(odd ? v[16 + k] : v[k]);
                  const float send = __uint_as_float(odd ? v[k] : v[16 + k]);
                  const float recv = __shfl_xor_sync(0xffffffffu, send, 1);
                  const float gate = odd ? recv : mine, up = odd ? mine : recv;
                  const int rr = c0 + (odd ? 16 : 0) + k;
                  if (rr < pc.crow && n < pc.N) M.mlp_act[(size_t)(pc.r0 + rr) * I + ii] = __float2bfloat16_rn(__fdividef(gate, 1.f + __expf(-gate)) * up);
                }
              }
            }
          }
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(tmem_empty_bar(buf));
          if (swiglu && !pc.final_ && pc.last_chunk) {   // publish this range's partial
            __threadfence();
            ptx::bar_sync(1, kLkEpiThreads);
            if (tid == 0) ptx::st_release_gpu(a.flag + (c.m * 2 + c.half) * (G / 2) + c.r, 1);
          }
          ++i;
          have = w.next(pc);
        }
        phase_arrive(p);
        if (dbg) dts[3 + 2 * p] = lk_now();
      } else {
        lk_fill_plane_counts(a.ph[a.ph[p].src], G / 2, tid, cnt_tab);   // before the wait: depends on the shapes only
        phase_wait(a.ph[p].src);
        if (dbg) dts[2 + 2 * p] = lk_now();
        if (type == LK_ROPE) lk_rope_phase(a, p, cta, G, tid, cnt_tab);
        else if (a.H <= 1024) lk_norm_phase<2>(a, p, cta, G, tid, red, cnt_tab);
        else if (a.H <= 2560) lk_norm_phase<5>(a, p, cta, G, tid, red, cnt_tab);
        else lk_norm_phase<8>(a, p, cta, G, tid, red, cnt_tab);       // H <= 4096 (tandem_init falls back to the separate kernels above that)
        phase_arrive(p);
        if (dbg) dts[3 + 2 * p] = lk_now();
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc_512(tmem_base);
}

// ---------------------------------------------------------------------------------------------- unit-test hook
// out[r, n] = sum over the partial planes of column block n / 256, in plane order (what the NORM / ROPE phases do)
__global__ void lk_sum_planes_kernel(const float* __restrict__ part, LkGeo g, int rows, int N, size_t stride, float* __restrict__ out) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)rows * N; i += (size_t)gridDim.x * blockDim.x) {
    const int n = (int)(i % N);
    const int cnt = lk_plane_count(g, n / kLkPairRows);
    float v = 0.f;
    for (int s = 0; s < cnt; ++s) v += part[s * stride + i];
    out[i] = v;
  }
}
// One GEMM phase of the layer kernel on its own: out = A W^T (fp32 [rows, N], planes summed here) or, swiglu, the bf16 SwiGLU
// activations [rows, N / 2]. pair = both models active (the same problem twice; model 1's result is returned), else one model
// (single-tile mode: every range is served by two CTAs, one per 128-row half). Synchronous. Returns 0 / -2 / -3 (abort flag: -4).
inline int lk_gemm_test(int rows, int N, int K, const void* A, const void* W, float* out, bool swiglu, bool pair) {
  if (rows <= 0) return 0;
  if (K % 8) return -1;
  int dev = 0, n_sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev);
  if (n_sms < 2) return -3;
  const int NR = n_sms / 2;
  TcGemmPlans* p = tc_gemm_create();
  if (!p) return -3;
  if (cudaFuncSetAttribute(layer_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLkSmemBytes) != cudaSuccess) { tc_gemm_destroy(p); return -3; }
  const LkGeo g = lk_geo(N, K, NR);
  const int planes = swiglu ? 1 : lk_max_planes(N, K, NR);
  const size_t cols = swiglu ? (size_t)NR * kLkPairRows : (size_t)planes * N;
  float* part[2] = {nullptr, nullptr}; bf16* act[2] = {nullptr, nullptr};
  int32_t* ints = nullptr; CUtensorMap* maps = nullptr;
  const size_t n_ints = 2 * C_NUM + kLkMaxPhases + 4 * NR + 1;
  int rc = 0;
  for (int m = 0; m < 2 && !rc; ++m) {
    if (cudaMalloc(&part[m], (size_t)rows * cols * 4) != cudaSuccess) rc = -2;
    if (!rc && swiglu && cudaMalloc(&act[m], (size_t)rows * (N / 2) * 2) != cudaSuccess) rc = -2;
  }
  if (!rc && cudaMalloc(&ints, n_ints * 4) != cudaSuccess) rc = -2;
  if (!rc && cudaMalloc(&maps, (size_t)(4 + 24) * sizeof(CUtensorMap)) != cudaSuccess) rc = -2;
  if (!rc) {
    std::vector<int32_t> hi(n_ints, 0);
    hi[C_ROWS] = pair ? rows : 0;              // model 0 is idle in the solo test, so that model 1 (the returned one) is the active one
    hi[C_NUM + C_ROWS] = rows;
    cudaMemcpy(ints, hi.data(), n_ints * 4, cudaMemcpyHostToDevice);
    std::vector<CUtensorMap> hm(4 + 24);
    for (int m = 0; m < 2; ++m) {
      for (int b = 0; b < 2; ++b) { const CUtensorMap* mp = tc_gemm_map(p, W, N, K, b == 0 ? kLkPairRows : kTcTileN); if (!mp) { rc = -3; break; } hm[m * 2 + b] = *mp; }
      for (int op = 0; op < 3 && !rc; ++op)
        for (int b = 0; b < 4; ++b) { const CUtensorMap* mp = tc_gemm_map(p, A, rows, K, 128 >> b); if (!mp) { rc = -3; break; } hm[4 + (op * 2 + m) * 4 + b] = *mp; }
    }
    cudaMemcpy(maps, hm.data(), hm.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice);
  }
  if (!rc) {
    LkArgs a{};
    a.ph[0] = LkPhase{swiglu ? LK_GEMM_SWIGLU : LK_GEMM_PARTIAL, N, K, 0, LK_A_ACT, -1, -1, 0};
    a.n_phases = 1;
    for (int m = 0; m < 2; ++m) { a.m[m].counts = ints + m * C_NUM; a.m[m].gemm_out = part[m]; a.m[m].mlp_act = act[m]; }
    a.H = N; a.row_cap = rows;
    a.bar = ints + 2 * C_NUM; a.flag = a.bar + kLkMaxPhases; a.abort_flag = a.flag + 4 * NR;
    a.wmaps = maps; a.amaps = maps + 4;
    if (launch_ex(layer_kernel, dim3(n_sms), dim3(kLkThreads), kLkSmemBytes, 0, false, a) != cudaSuccess) rc = -3;
    if (!rc && !swiglu) lk_sum_planes_kernel<<<296, 256>>>(part[1], g, rows, N, (size_t)rows * N, out);
    if (!rc && cudaDeviceSynchronize() != cudaSuccess) rc = -3;
    if (!rc && swiglu) cudaMemcpy(out, act[1], (size_t)rows * (N / 2) * 2, cudaMemcpyDeviceToDevice);
    int32_t ab = 0;
    if (!rc) { cudaMemcpy(&ab, a.abort_flag, 4, cudaMemcpyDeviceToHost); if (ab) rc = -4; }
  }
  for (int m = 0; m < 2; ++m) { if (part[m]) cudaFree(part[m]); if (act[m]) cudaFree(act[m]); }
  if (ints) cudaFree(ints);
  if (maps) cudaFree(maps);
  tc_gemm_destroy(p);
  cudaGetLastError();
  return rc;
}

// Timing hook: `iters` back-to-back single-phase launches for BOTH models (rows token rows each), every launch on different weight
// buffers (more than the L2 holds in total), between two CUDA events; mean milliseconds per launch.
inline int lk_gemm_time(int rows, int N, int K, int iters, bool swiglu, bool pdl, float* ms_out, int dbg_flags = 0) {
  int dev = 0, n_sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev);
  if (n_sms < 2 || (K % 8)) return -1;
  const int NR = n_sms / 2;
  TcGemmPlans* p = tc_gemm_create();
  if (!p) return -3;
  if (cudaFuncSetAttribute(layer_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLkSmemBytes) != cudaSuccess) { tc_gemm_destroy(p); return -3; }
  const size_t wbytes = (size_t)N * K * 2;
  const int nbuf = (int)std::min<size_t>(32, (400ull << 20) / wbytes + 2);   // model 0 uses buffer i, model 1 buffer i + 1
  const int planes = swiglu ? 1 : lk_max_planes(N, K, NR);
  const size_t cols = swiglu ? std::max((size_t)NR * kLkPairRows, (size_t)N / 2) : (size_t)planes * N;
  const size_t per_launch = kLkMaxPhases + 4 * NR;
  std::vector<void*> wb(nbuf, nullptr);
  void* A = nullptr; float* part[2] = {nullptr, nullptr}; bf16* act[2] = {nullptr, nullptr}; int32_t* ints = nullptr; CUtensorMap* maps = nullptr;
  const size_t n_ints = 2 * C_NUM + 1 + per_launch * (size_t)(nbuf + iters);
  int rc = 0;
  for (int i = 0; i < nbuf && !rc; ++i) { if (cudaMalloc(&wb[i], wbytes) != cudaSuccess) rc = -2; else cudaMemset(wb[i], 0x11, wbytes); }
  if (!rc && cudaMalloc(&A, (size_t)rows * K * 2) != cudaSuccess) rc = -2;
  for (int m = 0; m < 2 && !rc; ++m) {
    if (cudaMalloc(&part[m], (size_t)rows * cols * 4) != cudaSuccess) rc = -2;
    if (!rc && cudaMalloc(&act[m], (size_t)rows * (N / 2 + 8) * 2) != cudaSuccess) rc = -2;
  }
  if (!rc && cudaMalloc(&ints, n_ints * 4) != cudaSuccess) rc = -2;
  if (!rc && cudaMalloc(&maps, (size_t)(4 * nbuf + 24) * sizeof(CUtensorMap)) != cudaSuccess) rc = -2;
  if (!rc) {
    cudaMemset(A, 0x11, (size_t)rows * K * 2);
    std::vector<int32_t> hi(n_ints, 0);
    hi[C_ROWS] = rows; hi[C_NUM + C_ROWS] = rows;
    cudaMemcpy(ints, hi.data(), n_ints * 4, cudaMemcpyHostToDevice);
    std::vector<CUtensorMap> hm(4 * nbuf + 24);
    for (int i = 0; i < nbuf && !rc; ++i)
      for (int m = 0; m < 2; ++m)
        for (int b = 0; b < 2; ++b) {
          const CUtensorMap* mp = (dbg_flags & 2) ? tc_gemm_map(p, wb[(i + m) % nbuf], (int)((size_t)N * K / kTcBlockK), kTcBlockK, b == 0 ? kLkPairRows : kTcTileN)
                                                  : tc_gemm_map(p, wb[(i + m) % nbuf], N, K, b == 0 ? kLkPairRows : kTcTileN);
          if (!mp) { rc = -3; break; } hm[(i * 2 + m) * 2 + b] = *mp;
        }
    for (int op = 0; op < 3 && !rc; ++op)
      for (int m = 0; m < 2; ++m)
        for (int b = 0; b < 4; ++b) { const CUtensorMap* mp = tc_gemm_map(p, A, rows, K, 128 >> b); if (!mp) { rc = -3; break; } hm[4 * nbuf + (op * 2 + m) * 4 + b] = *mp; }
    cudaMemcpy(maps, hm.data(), hm.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice);
  }
  if (!rc) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int i = 0; i < nbuf + iters && !rc; ++i) {
      if (i == nbuf) cudaEventRecord(e0, 0);
      LkArgs a{};
      a.ph[0] = LkPhase{swiglu ? LK_GEMM_SWIGLU : LK_GEMM_PARTIAL, N, K, i % nbuf, LK_A_ACT, -1, -1, 0};
      a.n_phases = 1;
      for (int m = 0; m < 2; ++m) { a.m[m].counts = ints + m * C_NUM; a.m[m].gemm_out = part[m]; a.m[m].mlp_act = act[m]; }
      a.H = N; a.row_cap = rows;
      a.abort_flag = ints + 2 * C_NUM;
      a.bar = ints + 2 * C_NUM + 1 + per_launch * (size_t)i; a.flag = a.bar + kLkMaxPhases;
      a.wmaps = maps; a.amaps = maps + 4 * nbuf; a.dbg_flags = dbg_flags;
      if (launch_ex(layer_kernel, dim3(n_sms), dim3(kLkThreads), kLkSmemBytes, 0, pdl, a) != cudaSuccess) rc = -3;
    }
    cudaEventRecord(e1, 0);
    if (cudaDeviceSynchronize() != cudaSuccess) rc = -3;
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    *ms_out = ms / iters;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
  }
  for (void* b : wb) if (b) cudaFree(b);
  if (A) cudaFree(A);
  for (int m = 0; m < 2; ++m) { if (part[m]) cudaFree(part[m]); if (act[m]) cudaFree(act[m]); }
  if (ints) cudaFree(ints);
  if (maps) cudaFree(maps);
  tc_gemm_destroy(p);
  cudaGetLastError();
  return rc;
}

}  // namespace tandem
