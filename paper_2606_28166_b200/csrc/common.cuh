// common.cuh - shared device-side declarations of the tandem rollout engine (sm_100a).
// Notation follows DESIGN.md section 2: slot s = resident sequence, n_ctx = tokens in the shared context,
// ing[M] = context positions whose K/V model M has stored, row = one (sequence, position) processed this step.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace tandem {

constexpr int kPageTokens = 16;      // KV page size (BASELINE.json configs[2]: "paged KV with 16-token blocks")
constexpr int kAttnMinChunk = 256;   // smallest KV split of an attention item (models with few KV heads: the splits are the parallelism)
constexpr int kAttnMinChunkWide = 1024;   // ... with >= 8 KV heads (sequences x heads already fill the SMs; a short context in one piece needs no combine)
constexpr int kAttnMaxSplits = 4;    // an item is split along KV into at most this many chunks
constexpr int kAttnTileRows = 64;    // (query token, q-head of the group) rows per attention item = 4 MMA m-tiles
constexpr int kAttnSplitTiles = 4;   // sequences with at most this many q-tiles this step are also split along KV
// KV positions per split for a context of kv_len positions: a function of kv_len only, so the reduction order of a row
// never depends on what else is in the batch (batch invariance).
__host__ __device__ __forceinline__ int attn_chunk(int kv_len, int min_chunk) {
  const int c = ((kv_len + kAttnMaxSplits - 1) / kAttnMaxSplits + 63) & ~63;
  return c > min_chunk ? c : min_chunk;
}
constexpr int kMaxSlots = 1024;      // scheduler is one CTA with one thread per slot

typedef __nv_bfloat16 bf16;

template <typename T> struct Elem;
template <> struct Elem<float> {
  static __device__ __forceinline__ float ld(const float* p) { return *p; }
  static __device__ __forceinline__ void st(float* p, float v) { *p = v; }
};
template <> struct Elem<bf16> {
  static __device__ __forceinline__ float ld(const bf16* p) { return __bfloat162float(*p); }
  static __device__ __forceinline__ void st(bf16* p, float v) { *p = __float2bfloat16_rn(v); }
};

// 4 consecutive elements <-> 4 floats (16-byte fp32 / 8-byte bf16 accesses; pointers must be aligned accordingly)
__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 ld4(const bf16* p) {
  const uint2 t = *reinterpret_cast<const uint2*>(p);
  return make_float4(__uint_as_float(t.x << 16), __uint_as_float(t.x & 0xffff0000u), __uint_as_float(t.y << 16), __uint_as_float(t.y & 0xffff0000u));
}
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ void st4(bf16* p, float4 v) {
  const __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
  uint2 t; t.x = *reinterpret_cast<const uint32_t*>(&a); t.y = *reinterpret_cast<const uint32_t*>(&b);
  *reinterpret_cast<uint2*>(p) = t;
}
__device__ __forceinline__ float4 add4(float4 a, float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }

// Every kernel of the model chain is launched once for BOTH models (senior = 0, junior = 1): the two argument sets travel as
// one __grid_constant__ parameter and the model is a grid dimension (or, for attention, part of the unit index). Two
// independent half-sized problems per launch hide each other's latencies and halve the launch count.
template <typename A> struct Pair { A m[2]; };

// counts[] indices of a per-model step table
enum { C_ROWS = 0, C_SCHED = 1, C_EMIT = 2, C_ITEMS = 3, C_COMB = 4, C_PARTS = 5, C_NUM = 8 };

// Per-model tables the scheduler (S0) writes each step; everything downstream reads row counts from here,
// so every launch has a fixed grid and the whole step can be replayed as a CUDA graph.
struct StepTab {
  int32_t* counts;      // [C_NUM]
  int32_t* row_slot;    // [R] slot of the row's sequence
  int32_t* row_pos;     // [R] absolute position (kv_len of the row = pos + 1)
  int32_t* row_tok;     // [R] token id at that position
  int32_t* row_kvslot;  // [R] physical KV token index: page * kPageTokens + pos % kPageTokens
  int32_t* row_emit;    // [R] emit index j if this is the last row of a sequence that emits this step, else -1
  int32_t* emit_slot;   // [max_seqs] slot of emit index j
  // attention work items: item = n_tok consecutive rows of one sequence (one q-tile) x one KV range [kv0, kv1)
  int32_t* item_row0;   // [I] first row of the item
  int32_t* item_ntok;   // [I] rows (query tokens) in the item, <= tile_tok = kAttnTileRows / group
  int32_t* item_kv0;    // [I] first KV position of the item's range
  int32_t* item_kv1;    // [I] one past the last KV position (causal bound of the item's last row, or the split end)
  int32_t* item_part;   // [I] partial index of the item's first row (row j writes part + j), or -1: writes the final output
  int32_t* comb_row;    // [C] rows whose splits must be combined
  int32_t* comb_part0;  // [C] first partial of that row
  int32_t* comb_n;      // [C] number of partials
  int32_t* comb_stride; // [C] distance between consecutive partials of that row
  int32_t* comb_gpart;  // [C] one more partial of that row: its share of a shared-prefix run's item (share_prompt_pages = 2), or -1
};

struct SeqState {       // all [max_seqs]
  int32_t* seq_id; int32_t* prompt_len; int32_t* n_ctx; int32_t* ing[2]; int32_t* cap_c;
  int32_t* max_new; int32_t* n_emit; uint8_t* active; uint8_t* owner; uint8_t* done;
  int32_t* grp;         // prompt-sharing group of the sequence (index into GroupTab), -1 = none
};

struct PageTab {        // per model
  int32_t* bt;          // [max_seqs, max_pages] page ids
  int32_t* npages;      // [max_seqs]
  int32_t* free_pages;  // [pool_pages] stack of free page ids (page 0 is a dummy page, never handed out)
  int32_t* free_top;    // scalar: number of free pages on the stack
  int32_t* nshared;     // [max_seqs] leading entries of the sequence's block table that belong to its group (GroupTab), not to it
};

// Prompt-page sharing ("pages": the G rollouts of a GRPO group have identical prompts): the full pages of the
// common prompt are computed once per model - by the first member that runs that model, the donor - and referenced read-only from
// every member's block table. The group owns those pages; the last member to finish returns them. All [max_seqs] except pages.
struct GroupTab {
  int32_t* state[2];    // per model: 0 = nobody has started the shared prefix, 1 = the donor is ingesting it, 2 = pages[] valid
  int32_t* donor[2];    // slot of the donor while state == 1
  int32_t* pages[2];    // [max_seqs, max_pages] the group's page ids, npg[g] of them
  int32_t* npg;         // shared pages = floor((prompt_len - 1) / 16): every member keeps at least one prompt row of its own
  int32_t* ref;         // members that have not finished
};

struct DevStats {       // device-side accumulators (unsigned long long for atomicAdd)
  unsigned long long steps, tokens_emitted, rows[2], catchup_rows, kv_tokens_read, model_steps;
  unsigned long long shared_rows;   // prompt positions taken over from a group's shared pages instead of being recomputed
  unsigned long long starved;       // (sequence, step) pairs not scheduled because the model's page pool had no page left
  unsigned long long kv_tokens_shared;   // shared-prefix runs: KV positions the run's members after the first did not stream again
  int peak_pages_used[2]; int peak_resident; int err_oom;
};

struct StepIO {         // per-step optional outputs / overrides (device pointers, may be null)
  int32_t* token; uint8_t* owner; float* sen_logp; uint8_t* done; int32_t* argmax; int32_t* n_active;
  const int32_t* forced_tokens; long long forced_stride;
  const float* u_switch; long long u_switch_stride;
  const float* u_sample; long long u_sample_stride;
  float* dbg_logits;
};

struct RuleParams {
  float p; int switch_mode; int cap_k; float temperature; int eos_id; unsigned long long seed; float top_p; int top_k;
};

// ------------------------------------------------------------------------------------------------------------
// Counter-based generator (DESIGN.md section 3 R3). Philox-4x32-10 (Salmon et al., SC'11): written from the
// published round function; the oracle has its own NumPy implementation, the two share nothing.
__device__ __host__ __forceinline__ void philox_round(uint32_t c[4], uint32_t k0, uint32_t k1) {
  const uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
  const uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
  const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0;
  const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
  c[1] = (uint32_t)p1; c[3] = (uint32_t)p0; c[0] = n0; c[2] = n2;
}
__device__ __host__ __forceinline__ void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    philox_round(c, k0, k1);
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
}
// u = min((float(r) + 0.5f) * 2^-32, 1 - 2^-24), every operation rounded to nearest in fp32.
__device__ __forceinline__ float uniform_from_bits(uint32_t r) {
  float f = __uint2float_rn(r);
  f = __fadd_rn(f, 0.5f);
  f = __fmul_rn(f, 2.3283064365386963e-10f);   // 2^-32
  return fminf(f, 0.99999994f);                // 1 - 2^-24
}
__device__ __forceinline__ float u_switch_counter(unsigned long long seed, int seq_id, int t) {
  uint32_t c[4] = {0u, (uint32_t)t, (uint32_t)seq_id, 1u};
  philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
  return uniform_from_bits(c[0]);
}
// Gumbel variate from a uniform: E = -log1p(-u) (unit exponential), g = -ln E. Accurate libm calls, not intrinsics.
__device__ __forceinline__ float gumbel_from_uniform(float u) { return -logf(-log1pf(-u)); }

// Fused S8: what the LM head's epilogue keeps of a range of vocabulary ids for one emitting row (gemm_tcgen05.cuh, kTcEpiSample), and how
// two ranges combine. Symmetric (a + b == b + a bit for bit), ties go to the lower id: any merge tree gives the same ids, a fixed tree
// the same sums.
struct SamplePart { float m, s, gv, gz; int raw_id, g_id; };   // max z, sum exp((z - m) / T), best Gumbel-perturbed value and its z; argmax ids
__device__ __forceinline__ void sample_part_merge(SamplePart& a, const SamplePart& b, float inv_t) {
  const float mn = fmaxf(a.m, b.m);
  const float sa = a.m == -INFINITY ? 0.f : a.s * expf((a.m - mn) * inv_t), sb = b.m == -INFINITY ? 0.f : b.s * expf((b.m - mn) * inv_t);
  if (b.m > a.m || (b.m == a.m && b.raw_id < a.raw_id)) a.raw_id = b.raw_id;
  a.m = mn; a.s = sa + sb;
  if (b.gv > a.gv || (b.gv == a.gv && b.g_id < a.g_id)) { a.gv = b.gv; a.gz = b.gz; a.g_id = b.g_id; }
}

// ------------------------------------------------------------------------------------------------------------
// Programmatic dependent launch (PDL): a kernel launched with the attribute may start while its predecessor in the stream
// is still running; pdl_wait() blocks until the predecessor has completed and its writes are visible, pdl_trigger() lets
// the successor start launching. Both are no-ops in a kernel launched without the attribute. Rule used throughout: before
// pdl_wait() a kernel touches only constants (weights, tensor maps, the step tables written by the scheduler, which is
// never the direct predecessor) and its own shared memory / TMEM; every global write comes after it.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... P, typename... A>
inline cudaError_t launch_ex(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, A&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, P(args)...);
}
// the same with thread-block clusters of cluster_x CTAs along x (grid.x must be a multiple of it)
template <typename... P, typename... A>
inline cudaError_t launch_ex_cluster(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, int cluster_x, A&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = (unsigned)cluster_x; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, kernel, P(args)...);
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// Sum over a CTA of NT threads (NT multiple of 32, <= 1024); result broadcast to all threads. `red` >= 32 floats.
template <int NT> __device__ __forceinline__ float block_sum(float v, float* red) {
  v = warp_sum(v);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) red[w] = v;
  __syncthreads();
  float t = (l < NT / 32) ? red[l] : 0.f;
  return warp_sum(t);
}

}  // namespace tandem
