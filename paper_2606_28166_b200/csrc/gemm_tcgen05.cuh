// gemm_tcgen05.cuh - out[r, n] = sum_k A[r, k] W[n, k] for bf16 A, W with fp32 accumulation on the 5th-generation
// tensor cores (S3, S6, S7 and the LM head of the bf16 configs; BASELINE.json north_star (e)).
//
// Shape of the problem: W is [N, K] row-major (K contiguous), A is [rows, K] row-major, rows is small in decode
// (~64-256 per model per step) and only known on the device. So the kernel is "swap-AB": the weight tile is the
// M operand of tcgen05.mma (128 weight rows = 128 TMEM lanes) and the token rows are the N operand (32..256, a
// runtime field of the instruction descriptor), which makes ragged row counts free and turns the kernel into a
// weight streamer: every weight byte crosses HBM once (TMA, L2 evict-first), the activation tile is re-read from L2.
//   grid = (N/128 weight tiles, S K-splits); each CTA accumulates its K-slice for all rows in TMEM and writes an
//   fp32 partial out[s][r][n]; the consumer kernel sums the S partials in a fixed order (deterministic, no atomics).
//   warp 0: weight TMA   warp 6: activation TMA   warp 1: MMA issuer   warps 2-5, 7-10: epilogue (tcgen05.ld -> coalesced global
//   stores; two warps per TMEM lane quarter: the epilogue is an exposed tail, every CTA owns a single tile)
//   smem ring: stage = 16 KB of W (128 x 64 bf16, 128B swizzle) + 2 KB of A per 16 token rows (boxes of 128/64/32/16 rows), as many
//   stages as fit in 200 KB (4 at 256 rows, 6 at 128 rows, 10 at 32 rows).
// The gate/up projection of decode-sized steps and the LM head of the default sampling path have persistent kernels of their own
// (gemm_streamk.cuh, lmhead_sample.cuh); this kernel serves QKV, O, down, the materialised-logits LM head, scoring and prefill-sized launches.
#pragma once
#include <cuda.h>   // CUtensorMap and its enums only; the encode entry point is fetched at run time (no libcuda link)
#include <algorithm>
#include <map>
#include <vector>
#include <tuple>
#include "common.cuh"

namespace tandem {

constexpr int kTcTileN = 128;        // weight rows per CTA = UMMA M
constexpr int kTcBlockK = 64;        // bf16 elements per k-block = one 128-byte swizzle row
constexpr int kTcRowBox = 16;        // token rows per TMA box of A (= granularity of UMMA N)
constexpr int kTcMaxRows = 256;      // token rows per accumulator pass = max UMMA N
constexpr int kTcMaxStages = 10;
constexpr int kTcRingBytes = 200 * 1024;
constexpr int kTcSmemBytes = kTcRingBytes + 1024;   // + alignment slack
constexpr int kTcThreads = 352;        // warps: 0 weight TMA, 1 MMA, 2-5 and 7-10 epilogue (two per TMEM lane quarter), 6 activation TMA
constexpr int kTcWBytes = kTcTileN * kTcBlockK * 2;     // 16384
constexpr int kTcABoxBytes = kTcRowBox * kTcBlockK * 2; // 2048

// ---------------------------------------------------------------------------------------------- PTX wrappers
namespace ptx {
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar, uint64_t policy) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
               ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar), "l"(policy) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) { asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
template <int COLS> __device__ __forceinline__ void tmem_alloc(uint32_t smem_dst) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "n"(COLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int COLS> __device__ __forceinline__ void tmem_dealloc(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(COLS) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc], bf16 inputs, fp32 accumulate, one CTA.
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrives on the mbarrier once all previously issued tcgen05.mma of this thread have completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr));
}
// ---- CTA pair (cta_group::2): two CTAs of a cluster on the two SMs of a TPC drive one M = 256 MMA; each holds its own 128
// weight rows (A) and HALF of the token rows (B), so the activation bytes an SM has to pull out of L2 halve.
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t mapa_rank(uint32_t addr, uint32_t rank) {   // the same shared-memory offset in CTA `rank` of the cluster
  uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank)); return r;
}
__device__ __forceinline__ void mbar_expect_tx_cluster(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.release.cluster.shared::cluster.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar) : "memory");
}
// TMA load into this CTA's shared memory that signals a barrier which may live in the peer CTA of the pair
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar_cluster, uint64_t policy) {
  asm volatile("cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
               ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar_cluster), "l"(policy) : "memory");
}
template <int COLS> __device__ __forceinline__ void tmem_alloc_pair(uint32_t smem_dst) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "n"(COLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
template <int COLS> __device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(COLS) : "memory");
}
__device__ __forceinline__ void umma_bf16_pair(uint32_t d_tmem, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrives on the barrier at this shared-memory offset in BOTH CTAs of the pair once the MMAs issued so far have completed
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr));
}
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
// the same with an immediate barrier id: ptxas then reserves only the barriers a kernel names (a register id makes it reserve all
// 16, and two CTAs per SM no longer fit)
template <int ID> __device__ __forceinline__ void bar_sync_id(int n) { asm volatile("bar.sync %0, %1;" ::"n"(ID), "r"(n) : "memory"); }
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// One lane of a converged warp. The TMA / MMA warps run their loops with all 32 lanes and issue under elect_one(): the operands
// (descriptors, addresses) are then provably warp-uniform and stay in uniform registers. Issued from a single divergent thread
// (`if (lane == 0)`), every tcgen05.mma cost 151 cycles (R2UR moves) instead of 99 / 128 at N <= 128 / N = 256 (measured, B200).
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(p));
  return p != 0;
}
}  // namespace ptx

// Shared-memory matrix descriptor of a K-major bf16 tile whose rows are 128 bytes (64 elements) with the 128-byte
// swizzle TMA wrote: 8-row groups are 1024 bytes apart (SBO), descriptor version 1 (sm_100), layout type 2.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);        // start address, bits [0,14)
  d |= (uint64_t)1 << 16;                              // leading byte offset (unused for swizzled K-major), bits [16,30)
  d |= (uint64_t)(1024u >> 4) << 32;                   // stride byte offset, bits [32,46)
  d |= (uint64_t)1 << 46;                              // version
  d |= (uint64_t)2 << 61;                              // SWIZZLE_128B
  return d;
}
// Instruction descriptor, kind::f16: D fp32, A and B bf16, both K-major, M = 128, N = n (multiple of 16, <= 256).
__device__ __forceinline__ uint32_t umma_idesc_bf16(int n, int m = kTcTileN) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}


struct TcMaps { CUtensorMap w[2], a[2][4]; };   // per model: weight descriptor; activation descriptors with 128/64/32/16-row boxes

struct TcGemmArgs {
  float* out;                 // [n_split][row_cap][N] fp32 partials
  const int32_t* rows_ptr;    // device scalar with the live row count, or null
  int rows_fixed;
  int N, K, n_split;
  size_t split_stride;        // floats between partials
  int ring_bytes;             // shared-memory ring of this launch (200 KB: one CTA per SM; 98 KB: two)
  int chunk_grid;             // >= 1: the 256-row chunks of the token rows are dealt round-robin to this many CTAs per (tile, split)
                              // (gridDim.y = n_split * chunk_grid); 1 = one CTA walks all chunks
  // kTcEpiSample (lmhead_sample_kernel: the LM head of the default sampling path, S8): the logits never reach HBM
  const int32_t* emit_slot;   // [rows] slot of emitting row j
  const int32_t* n_emit;      // [max_seqs] tokens emitted so far (t = n_emit + 1 addresses the uniforms)
  const int32_t* seq_id;      // [max_seqs]
  float inv_t; int greedy; uint32_t key0, key1;   // 1 / temperature (1 if greedy), Philox key = seed
};
constexpr int kTcSampleVals = 8;       // floats per (weight tile, row) partial: max z, sum exp, raw best id, Gumbel best value, its id, its z, 2 spare

// ---------------------------------------------------------------------------------------------- the kernel
enum { kTcEpiPartial = 0, kTcEpiSwiGLU = 1, kTcEpiSample = 2 };

// EPI  = kTcEpiPartial: fp32 partial out[split][r][n];
//        kTcEpiSwiGLU : W rows interleaved (2i = gate_i, 2i+1 = up_i), n_split = 1: act[r][i] = silu(gate) * up as bf16.
// (kTcEpiSample, the LM head of the default sampling path with S8's reductions in its epilogue, is a kernel of its own:
//  lmhead_sample.cuh - persistent, two TMEM accumulators.)
// Cluster launches with TMA multicast of the activation boxes (2 and 4 CTAs) were built and measured: no gain at any of
// the projection shapes on B200 (profiles/gemm_sweep_r1.md): multicast does not lower what each SM has to ingest. The CTA pair does.
// PAIR = true: launched in clusters of two CTAs along x (adjacent weight tiles). The pair runs one cta_group::2 MMA with M = 256:
//        each CTA streams its own 128 weight rows and HALF of the token rows, both signal the leader's (rank 0) full barrier,
//        the leader's MMA warp issues for both and its commits arrive on the empty / accumulator barriers of both CTAs; each CTA
//        drains its own 128 TMEM lanes. The activation bytes an SM pulls out of L2 halve (profiles/gemm_sweep_r1.md: the
//        projections are bound by SM ingest, not HBM, above ~64 token rows).
template <int EPI, bool PAIR>
__global__ void __launch_bounds__(kTcThreads, 2)   // two CTAs per SM whenever the ring allows: <= 93 registers per thread
gemm_tcgen05_kernel(const __grid_constant__ TcMaps maps, const __grid_constant__ Pair<TcGemmArgs> gp) {
  const TcGemmArgs& g = gp.m[blockIdx.z];                  // blockIdx.z = model
  const CUtensorMap* tmap_w = &maps.w[blockIdx.z];
  const CUtensorMap* tmap_a = maps.a[blockIdx.z];
  extern __shared__ uint8_t tc_smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * kTcMaxStages + 2];
  __shared__ uint32_t tmem_base_smem;

  pdl_trigger();
  const int rows = g.rows_ptr ? *g.rows_ptr : g.rows_fixed;   // scheduler output: complete before any kernel of the chain starts
  if (rows <= 0) { pdl_wait(); return; }                   // uniform over the grid: nothing was scheduled for this model
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = PAIR ? ptx::cluster_ctarank() : 0u;
  const bool leader = rank == 0;
  const int n0 = blockIdx.x * kTcTileN;
  const int split = (int)blockIdx.y % g.n_split;
  const int cslice = (int)blockIdx.y / g.n_split, cstep = g.chunk_grid;   // this CTA's chunks: cslice, cslice + cstep, ...
  const int kb_total = (g.K + kTcBlockK - 1) / kTcBlockK;
  const int kb0 = (int)((long long)kb_total * split / g.n_split);
  const int kb1 = (int)((long long)kb_total * (split + 1) / g.n_split);
  const int n_chunks = (rows + kTcMaxRows - 1) / kTcMaxRows;
  // token rows of a chunk are padded to the box granularity; a pair splits them in two halves of whole boxes
  constexpr int kPad = PAIR ? 2 * kTcRowBox : kTcRowBox;
  auto chunk_cols = [&](int r0) { return ((min(rows - r0, kTcMaxRows) + kPad - 1) / kPad) * kPad; };
  const int nbox_max = chunk_cols(0) / kTcRowBox / (PAIR ? 2 : 1);   // boxes this CTA loads per stage
  const int stage_bytes = kTcWBytes + nbox_max * kTcABoxBytes;
  const int n_stages = min(kTcMaxStages, g.ring_bytes / stage_bytes);

  const uint32_t ring = (ptx::smem_u32(tc_smem_raw) + 1023u) & ~1023u;   // 128B swizzle atoms are 1024-byte aligned
  const uint32_t bar0 = ptx::smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (uint32_t)(kTcMaxStages + s); };
  const uint32_t tmem_full_bar = bar0 + 8u * (2 * kTcMaxStages);
  const uint32_t tmem_empty_bar = tmem_full_bar + 8u;

  if (threadIdx.x == 0) {
    // full: weight + activation producers (a pair: the leader's two, which also post the peer's bytes); empty / accumulator-full: one commit
    for (int s = 0; s < n_stages; ++s) { ptx::mbar_init(full_bar(s), 2); ptx::mbar_init(empty_bar(s), 1); }
    ptx::mbar_init(tmem_full_bar, 1);
    ptx::mbar_init(tmem_empty_bar, PAIR ? 16 : 8);         // the epilogue warps (of both CTAs; only the leader's is used)
    ptx::fence_mbar_init();
    ptx::prefetch_tmap(tmap_w);
    ptx::prefetch_tmap(tmap_a);
  }
  if (warp == 2) { if (PAIR) ptx::tmem_alloc_pair<kTcMaxRows>(ptx::smem_u32(&tmem_base_smem)); else ptx::tmem_alloc<kTcMaxRows>(ptx::smem_u32(&tmem_base_smem)); }
  ptx::tc_fence_before();
  if (PAIR) ptx::cluster_sync_all(); else __syncthreads();   // barriers of both CTAs are initialised before anyone signals them
  ptx::tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  if (warp == 0) {
    // ===== weight producer: weights stream once (L2 evict-first) and do not depend on the predecessor kernel, so this
    // warp never waits for it. (A thread issues one TMA box in ~0.1-0.2 us: weights and activations have a warp each.)
    {
      const uint64_t pol_w = ptx::policy_evict_first();
      int it = 0;
      for (int c = cslice; c < n_chunks; c += cstep)
        for (int kb = kb0; kb < kb1; ++kb, ++it) {
          const int s = it % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(it / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            if (PAIR) {   // the leader posts the bytes of both CTAs' loads (a remote arrive per stage would stall the peer's producer)
              if (leader) ptx::mbar_expect_tx(full_bar(s), 2u * (uint32_t)kTcWBytes);
              ptx::tma_load_2d_pair(ring + (uint32_t)(s * stage_bytes), tmap_w, kb * kTcBlockK, n0, ptx::mapa_rank(full_bar(s), 0), pol_w);
            } else {
              ptx::mbar_expect_tx(full_bar(s), (uint32_t)kTcWBytes);
              ptx::tma_load_2d(ring + (uint32_t)(s * stage_bytes), tmap_w, kb * kTcBlockK, n0, full_bar(s), pol_w);
            }
          }
          __syncwarp();
        }
    }
  } else if (warp == 6) {
    // ===== activation producer: the activation tile is shared by every CTA (L2 evict-last); greedy 128/64/32/16-row boxes
    {
      const uint64_t pol_a = ptx::policy_evict_last();
      pdl_wait();                                            // the activations come from the predecessor kernel
      int it = 0;
      for (int c = cslice; c < n_chunks; c += cstep) {
        const int cols = chunk_cols(c * kTcMaxRows);
        const int nbox = cols / kTcRowBox / (PAIR ? 2 : 1);
        const int r0 = c * kTcMaxRows + (PAIR ? (int)rank * (cols / 2) : 0);   // a pair: this CTA's half of the token rows
        for (int kb = kb0; kb < kb1; ++kb, ++it) {
          const int s = it % n_stages;
          ptx::mbar_wait(empty_bar(s), ((uint32_t)(it / n_stages) & 1u) ^ 1u);
          if (ptx::elect_one()) {
            const uint32_t fb = PAIR ? ptx::mapa_rank(full_bar(s), 0) : full_bar(s);
            if (!PAIR) ptx::mbar_expect_tx(fb, (uint32_t)(nbox * kTcABoxBytes));
            else if (leader) ptx::mbar_expect_tx(full_bar(s), 2u * (uint32_t)(nbox * kTcABoxBytes));
            const uint32_t dst = ring + (uint32_t)(s * stage_bytes) + kTcWBytes;
            int j = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              const int bx = 8 >> b;
              while (nbox - j >= bx) {
                if (PAIR) ptx::tma_load_2d_pair(dst + j * kTcABoxBytes, tmap_a + b, kb * kTcBlockK, r0 + j * kTcRowBox, fb, pol_a);
                else ptx::tma_load_2d(dst + j * kTcABoxBytes, tmap_a + b, kb * kTcBlockK, r0 + j * kTcRowBox, fb, pol_a);
                j += bx;
              }
            }
          }
          __syncwarp();
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: one elected lane drives the tensor core for the whole CTA (for both CTAs of a pair: the leader's)
    if (leader) {
      int it = 0;
      for (int c = cslice, ci = 0; c < n_chunks; c += cstep, ++ci) {
        const int ncols = chunk_cols(c * kTcMaxRows);
        const uint32_t idesc = umma_idesc_bf16(ncols, PAIR ? 2 * kTcTileN : kTcTileN);
        ptx::mbar_wait(tmem_empty_bar, ((uint32_t)ci & 1u) ^ 1u);
        ptx::tc_fence_after();
        for (int kb = kb0; kb < kb1; ++kb, ++it) {
          const int s = it % n_stages;
          const uint32_t ph = (uint32_t)(it / n_stages) & 1u;
          ptx::mbar_wait(full_bar(s), ph);
          ptx::tc_fence_after();
          const uint32_t sw = ring + (uint32_t)(s * stage_bytes);
          const uint64_t dw = umma_desc_sw128(sw), da = umma_desc_sw128(sw + kTcWBytes);
          if (ptx::elect_one()) {
#pragma unroll
            for (int k = 0; k < kTcBlockK / 16; ++k) {   // UMMA K = 16 bf16 = 32 bytes: advance the start address inside the swizzle row
              if (PAIR) ptx::umma_bf16_pair(tmem_base, dw + (uint64_t)(2 * k), da + (uint64_t)(2 * k), idesc, (kb > kb0 || k > 0) ? 1u : 0u);
              else ptx::umma_bf16(tmem_base, dw + (uint64_t)(2 * k), da + (uint64_t)(2 * k), idesc, (kb > kb0 || k > 0) ? 1u : 0u);
            }
            if (PAIR) ptx::umma_commit_pair(empty_bar(s)); else ptx::umma_commit(empty_bar(s));   // stage free once these MMAs have read it
          }
          __syncwarp();
        }
        if (ptx::elect_one()) { if (PAIR) ptx::umma_commit_pair(tmem_full_bar); else ptx::umma_commit(tmem_full_bar); }   // accumulator of this chunk complete
        __syncwarp();
      }
    }
  } else {
    // ===== epilogue: warp w may touch TMEM lanes 32*(w%4)..+31; lane = weight row n, column = token row r. Each lane quarter
    // has two warps (2-5 and 7-10) that take alternate groups of 32 columns.
    const int q = warp & 3;
    const int half = warp >= 7 ? 1 : 0;
    const int n = n0 + q * 32 + lane;
    float* outp = g.out + (size_t)split * g.split_stride;
    const uint32_t te_bar = PAIR ? ptx::mapa_rank(tmem_empty_bar, 0) : tmem_empty_bar;
    pdl_wait();                                            // the predecessor may still be reading the buffer this kernel writes
    for (int c = cslice, ci = 0; c < n_chunks; c += cstep, ++ci) {
      const int r0 = c * kTcMaxRows;
      const int crow = min(rows - r0, kTcMaxRows);
      ptx::mbar_wait(tmem_full_bar, (uint32_t)ci & 1u);
      ptx::tc_fence_after();
      for (int c0 = 32 * half; c0 < crow; c0 += 64) {
        uint32_t v[32];
        ptx::tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)c0, v);
        ptx::tmem_ld_wait();
        if (EPI == kTcEpiPartial) {
          if (n < g.N) {
#pragma unroll
            for (int j = 0; j < 32; ++j)
              if (c0 + j < crow) outp[(size_t)(r0 + c0 + j) * g.N + n] = __uint_as_float(v[j]);
          }
        } else {
          // even lane = gate row i, odd lane = up row i of the same intermediate index i: swap halves of the 32 columns so
          // that the even lane finishes columns [0,16) and the odd lane columns [16,32)
          const bool odd = lane & 1;
          const int i = n >> 1, I = g.N >> 1;
          bf16* act = reinterpret_cast<bf16*>(g.out);
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const float mine = __uint_as_float(odd ? v[16 + j] : v[j]);
            const float send = __uint_as_float(odd ? v[j] : v[16 + j]);
            const float recv = __shfl_xor_sync(0xffffffffu, send, 1);
            const float gate = odd ? recv : mine, up = odd ? mine : recv;
            const int r = c0 + (odd ? 16 : 0) + j;
            if (r < crow && n < g.N) act[(size_t)(r0 + r) * I + i] = __float2bfloat16_rn(__fdividef(gate, 1.f + __expf(-gate)) * up);   // bf16 result: fast exp / divide are exact enough
          }
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) { if (PAIR) ptx::mbar_arrive_cluster(te_bar); else ptx::mbar_arrive(te_bar); }
    }
  }
  ptx::tc_fence_before();
  if (PAIR) ptx::cluster_sync_all(); else __syncthreads();   // a pair: neither CTA leaves while the other may still read its shared memory / signal it
  if (warp == 2) { if (PAIR) ptx::tmem_dealloc_pair<kTcMaxRows>(tmem_base); else ptx::tmem_dealloc<kTcMaxRows>(tmem_base); }
}

#include "lmhead_sample.cuh"   // lmhead_sample_kernel (kTcEpiSample); needs everything above

// ---------------------------------------------------------------------------------------------- host side
// K-splits: as many as keep the whole launch (all tiles of all models in it) within one CTA per SM, each slice >= 4 k-blocks.
// One CTA per SM with the deep 200 KB ring beats two per SM with an uneven second layer (measured on the 4B shape, both models
// per launch: O and down 3 splits = 120 CTAs: 12.98 ms per step; 4 splits = 160 CTAs: 13.13; 7 splits = 280 CTAs: 13.15), and
// the consumer kernel has fewer partials to sum. A function of the shape and of the number of models per launch only, so the
// reduction order (and every logit) is independent of the batch.
inline int tc_gemm_splits(int N, int K, int n_models = 1, int n_sms = 148) {
  const int tiles = n_models * ((N + kTcTileN - 1) / kTcTileN), kb = (K + kTcBlockK - 1) / kTcBlockK;
  int s = 1;
  while (tiles * (s + 1) <= n_sms && (s + 1) * 4 <= kb && s < 16) ++s;
  return s;
}

typedef CUresult (*TcEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcGemmPlans {
  TcEncodeFn encode = nullptr;
  std::map<std::tuple<const void*, int, int, int>, CUtensorMap> maps;   // (base, rows, K, box_rows) -> descriptor
};

inline TcGemmPlans* tc_gemm_create() {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn || q != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  bool ok = true;
  ok &= cudaFuncSetAttribute(gemm_tcgen05_kernel<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes) == cudaSuccess;
  ok &= cudaFuncSetAttribute(gemm_tcgen05_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes) == cudaSuccess;
  ok &= cudaFuncSetAttribute(lmhead_sample_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLmSmemBytes) == cudaSuccess;
  ok &= cudaFuncSetAttribute(gemm_tcgen05_kernel<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes) == cudaSuccess;
  ok &= cudaFuncSetAttribute(gemm_tcgen05_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    return nullptr;
  }
  TcGemmPlans* p = new TcGemmPlans();
  p->encode = (TcEncodeFn)fn;
  return p;
}
inline void tc_gemm_destroy(TcGemmPlans* p) { delete p; }
inline void tc_gemm_invalidate(TcGemmPlans* p, int) { if (p) p->maps.clear(); }

// Descriptor of a row-major bf16 matrix [n_rows, K] tiled in boxes of box_rows x 64 elements, 128-byte swizzle;
// out-of-bounds elements read as zero (ragged K tails and row tails need no special case).
inline const CUtensorMap* tc_gemm_map(TcGemmPlans* p, const void* base, int n_rows, int K, int box_rows) {
  auto key = std::make_tuple(base, n_rows, K, box_rows);
  auto it = p->maps.find(key);
  if (it != p->maps.end()) return &it->second;
  CUtensorMap m;
  const cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)n_rows};
  const cuuint64_t strides[1] = {(cuuint64_t)K * 2};
  const cuuint32_t box[2] = {(cuuint32_t)kTcBlockK, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = p->encode(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return nullptr;
  return &(p->maps[key] = m);
}

// Descriptor of a q buffer [n_rows][n_heads][D] bf16 in boxes of tok_box tokens x G heads x 64 elements (one 64-dim half of an attention
// q-tile whose rows are (token, head of the group) pairs), 128-byte swizzle; rows beyond n_rows read as zero.
inline bool tc_map_q3d(TcGemmPlans* p, CUtensorMap* out, const void* base, int D, int n_heads, int n_rows, int G, int tok_box) {
  const cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)n_heads, (cuuint64_t)n_rows};
  const cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)n_heads * D * 2};
  const cuuint32_t box[3] = {64u, (cuuint32_t)G, (cuuint32_t)tok_box};
  const cuuint32_t estr[3] = {1, 1, 1};
  return p->encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Launch on `s`. out receives *n_split partials, *split_stride floats apart (epi = kTcEpiPartial), or the bf16 SwiGLU
// activations [rows, N/2] (epi = kTcEpiSwiGLU; W rows interleaved gate/up). Returns 0, or -1 (TANDEM_EINVAL) / -3 (TANDEM_ECUDA).
// which == 4 (LM head) never splits: the sampler reads the logits in place.
template <int EPI>
inline int tc_gemm_launch_epi(const TcMaps& maps, const Pair<TcGemmArgs>& g, dim3 grid, cudaStream_t s, bool pdl, bool pair) {
  const size_t smem = (size_t)g.m[0].ring_bytes + 1024;
  if (pair) return launch_ex_cluster(gemm_tcgen05_kernel<EPI, true>, grid, dim3(kTcThreads), smem, s, pdl, 2, maps, g) == cudaSuccess ? 0 : -3;
  return launch_ex(gemm_tcgen05_kernel<EPI, false>, grid, dim3(kTcThreads), smem, s, pdl, maps, g) == cudaSuccess ? 0 : -3;
}
struct TcSampleCfg { const int32_t* emit_slot[2]; const int32_t* n_emit; const int32_t* seq_id; float inv_t; int greedy; unsigned long long seed; };
struct TcGemmTune { int ring_kb = 0, splits = 0; bool pdl = false; int pair = 0; int chunk_grid = 1; int n_sms = 148; const TcSampleCfg* sample = nullptr; };   // pair: 1 = CTA pairs (cta_group::2), 0 = single CTAs   // 0 = automatic; overrides for tuning / tandem_test_gemm_time
// One launch for n_models (1 or 2) problems of the same shape: out[m] = A[m] W[m]^T, rows of model m from rows_ptr[m].
inline int tc_gemm_launch(TcGemmPlans* p, int n_models, int which, const void* const* A, const void* const* W, int N, int K, float* const* out,
                          const int32_t* const* rows_ptr, int rows_cap, int* n_split, size_t* split_stride, cudaStream_t s, int epi = kTcEpiPartial,
                          const TcGemmTune* tune = nullptr) {
  if (!p || (K % 8) != 0) return -1;                       // TMA needs 16-byte row strides
  const int n_sms = tune ? tune->n_sms : 148;
  int S = (which == 4 || epi != kTcEpiPartial) ? 1 : tc_gemm_splits(N, K, n_models, n_sms);
  if (tune && tune->splits > 0) S = tune->splits;
  *n_split = S;
  *split_stride = (size_t)rows_cap * N;
  const int tiles = (N + kTcTileN - 1) / kTcTileN;
  const bool pair = tune && tune->pair > 0;
  const int tiles_pad = pair ? (tiles + 1) & ~1 : tiles;   // a pair takes two adjacent weight tiles (a tile past N reads zeros and writes nothing)
  TcMaps maps;
  Pair<TcGemmArgs> g;
  // many token rows (scoring, prefill): the 256-row chunks go to different CTAs, so the launch has more and shorter CTAs and a
  // shorter tail (ncu, 512 rows, gate/up as 304 CTAs on 296 slots: SMs active 60% of the kernel's duration)
  const int CG = (tune && tune->chunk_grid > 1) ? std::min(tune->chunk_grid, (rows_cap + kTcMaxRows - 1) / kTcMaxRows) : 1;
  const int ring = (tune && tune->ring_kb > 0) ? tune->ring_kb * 1024
                                                : (tiles_pad * S * CG * n_models > n_sms ? 109 * 1024 : kTcRingBytes);   // more CTAs than SMs: two share an SM
  for (int m = 0; m < 2; ++m) {
    const int mm = m < n_models ? m : 0;
    const CUtensorMap* mw = tc_gemm_map(p, W[mm], N, K, kTcTileN);
    if (!mw) return -3;
    maps.w[m] = *mw;
    for (int b = 0; b < 4; ++b) {
      const CUtensorMap* ma = tc_gemm_map(p, A[mm], rows_cap, K, 128 >> b);
      if (!ma) return -3;
      maps.a[m][b] = *ma;
    }
    g.m[m] = TcGemmArgs{out[mm], rows_ptr ? rows_ptr[mm] : nullptr, rows_cap, N, K, S, *split_stride,
                        epi == kTcEpiSample ? kLmRingBytes : ring, CG, nullptr, nullptr, nullptr, 1.f, 1, 0u, 0u};
    if (epi == kTcEpiSample) {
      if (!tune || !tune->sample) return -1;
      const TcSampleCfg& sc = *tune->sample;
      g.m[m].emit_slot = sc.emit_slot[mm]; g.m[m].n_emit = sc.n_emit; g.m[m].seq_id = sc.seq_id; g.m[m].inv_t = sc.inv_t; g.m[m].greedy = sc.greedy;
      g.m[m].key0 = (uint32_t)sc.seed; g.m[m].key1 = (uint32_t)(sc.seed >> 32);
    }
  }
  dim3 grid(tiles_pad, S * CG, n_models);
  const bool pdl = tune && tune->pdl;
  if (epi == kTcEpiSwiGLU) return tc_gemm_launch_epi<1>(maps, g, grid, s, pdl, pair);
  if (epi == kTcEpiSample)   // persistent: one CTA per SM walks the (weight tile, model) units
    return launch_ex(lmhead_sample_kernel, dim3(std::min(n_sms, tiles * n_models)), dim3(kLmThreads), (size_t)kLmSmemBytes, s, pdl, maps, g) == cudaSuccess ? 0 : -3;
  return tc_gemm_launch_epi<0>(maps, g, grid, s, pdl, pair);
}

// Unit-test hook: out[rows, N] = A W^T (partials summed here), synchronous.
__global__ void tc_sum_partials_kernel(const float* __restrict__ part, int n_split, size_t stride, float* __restrict__ out, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    float v = 0.f;
    for (int s = 0; s < n_split; ++s) v += part[s * stride + i];
    out[i] = v;
  }
}
inline int tc_gemm_test(int rows, int N, int K, const void* A, const void* W, float* out, int epi = kTcEpiPartial, bool pair = false) {
  TcGemmTune tune; tune.pair = pair ? 1 : 0;
  if (rows == 0) return 0;
  TcGemmPlans* p = tc_gemm_create();
  if (!p) return -3;
  if (epi == kTcEpiSwiGLU) {   // W rows interleaved gate/up; out is bf16 [rows, N/2]
    int ns; size_t ss;
    int rc = tc_gemm_launch(p, 1, 2, &A, &W, N, K, &out, nullptr, rows, &ns, &ss, 0, epi, &tune);
    if (rc == 0) rc = cudaDeviceSynchronize() == cudaSuccess ? 0 : -3;
    tc_gemm_destroy(p);
    return rc;
  }
  const int S = tc_gemm_splits(N, K);
  float* part = nullptr;
  if (cudaMalloc(&part, (size_t)S * rows * N * sizeof(float)) != cudaSuccess) { tc_gemm_destroy(p); return -2; }
  int ns; size_t ss;
  int rc = tc_gemm_launch(p, 1, 0, &A, &W, N, K, &part, nullptr, rows, &ns, &ss, 0, kTcEpiPartial, &tune);
  if (rc == 0) {
    tc_sum_partials_kernel<<<296, 256>>>(part, ns, ss, out, (size_t)rows * N);
    rc = cudaDeviceSynchronize() == cudaSuccess ? 0 : -3;
  }
  cudaFree(part);
  tc_gemm_destroy(p);
  return rc;
}

// Timing hook: `iters` back-to-back launches of the [rows, K] x [N, K]^T GEMM, each on a different weight buffer (enough
// buffers to exceed the L2), between two CUDA events; returns the mean milliseconds per launch.
inline int tc_gemm_time(int rows, int N, int K, int iters, const TcGemmTune& tune, int epi, float* ms_out) {
  TcGemmPlans* p = tc_gemm_create();
  if (!p) return -3;
  const size_t wbytes = (size_t)N * K * 2;
  const int nbuf = (int)std::min<size_t>(64, (400ull << 20) / wbytes + 2);
  std::vector<void*> wb(nbuf, nullptr);
  void* A = nullptr; float* out = nullptr;
  int rc = 0;
  const int S = tune.splits > 0 ? tune.splits : tc_gemm_splits(N, K);
  for (int i = 0; i < nbuf && !rc; ++i) { if (cudaMalloc(&wb[i], wbytes) != cudaSuccess) rc = -2; else cudaMemset(wb[i], 0x11, wbytes); }
  if (!rc && cudaMalloc(&A, (size_t)rows * K * 2) != cudaSuccess) rc = -2;
  if (!rc && cudaMalloc(&out, (size_t)S * rows * N * 4) != cudaSuccess) rc = -2;
  if (!rc) {
    cudaMemset(A, 0x11, (size_t)rows * K * 2);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    int ns; size_t ss;
    for (int i = 0; i < nbuf + iters && !rc; ++i) {
      if (i == nbuf) cudaEventRecord(e0, 0);
      const void* Ap = A; const void* Wp = wb[i % nbuf];
      rc = tc_gemm_launch(p, 1, epi == kTcEpiSwiGLU ? 2 : 0, &Ap, &Wp, N, K, &out, nullptr, rows, &ns, &ss, 0, epi, &tune);
    }
    cudaEventRecord(e1, 0);
    if (cudaDeviceSynchronize() != cudaSuccess) rc = -3;
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    *ms_out = ms / iters;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
  }
  for (void* b : wb) if (b) cudaFree(b);
  if (A) cudaFree(A);
  if (out) cudaFree(out);
  tc_gemm_destroy(p);
  cudaGetLastError();
  return rc;
}

}  // namespace tandem
