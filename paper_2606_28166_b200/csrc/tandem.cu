// tandem.cu - host side of the C ABI declared in include/tandem.h: handle, weights, admission, the step
// (S0 scheduler -> S1..S8 for both models, every kernel launched once for the pair -> finalize) and whole-rollout generation. All arithmetic of the path
// runs in the kernels of this directory; there is no CPU fallback.
#include "../../include/tandem.h"
#include "../../include/tandem_test.h"

#include <cuda_runtime.h>
#include <cuda_bf16.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <mutex>
#include <vector>

#include "common.cuh"
#include "kernels.cuh"
#include "attention.cuh"
#include "attention_mma.cuh"
#include "attention_tcgen05.cuh"
#include "gemm_simt.cuh"
#include "gemm_tcgen05.cuh"
#include "gemm_streamk.cuh"
#include "grpo.cuh"

using namespace tandem;
constexpr int kSampleMaxChunks = 32;

namespace {

struct ModelWeights {
  bool loaded = false;
  void *embed = nullptr, *lm_head = nullptr, *final_norm = nullptr;
  std::vector<void*> attn_norm, wqkv, wo, mlp_norm, wgu, wdown;
};

struct Workspace {  // per model, sized for row_cap rows
  float* x = nullptr;          // residual stream fp32 [R, H]
  void* act = nullptr;         // normalised activations (GEMM A operand) [R, H]
  void* q = nullptr;           // RoPE'd queries [R, nq*d]: fp32 (ALU attention) or bf16 (tensor-core attention)
  void* attn_out = nullptr;    // [R, nq*d]
  void* mlp_act = nullptr;     // silu(gate)*up [R, I]
  void* lm_in = nullptr;       // final-normed last rows [max_seqs, H]
  float* gemm_out = nullptr;   // split-K partial outputs [S][R][N], S*N <= gemm_out_cols
  float* logits = nullptr;     // [max_seqs, V]
  void* score_lm_in = nullptr; float* score_logits = nullptr;   // tandem_score: [row_cap, H] and [row_cap, V], allocated at its first call
  float* chunk_part = nullptr; int32_t* chunk_ctr = nullptr;   // sampler: per-slice partials and arrival counters
  float* spart = nullptr;      // fused S8: the LM head's per-(row, weight tile) sampling partials [max_seqs][V / 128][8]
  float* part_acc = nullptr; float2* part_ml = nullptr;
  void* kv = nullptr;          // page pool: [layer][K|V][page][nkv][16][d]
  int32_t* tab_mem = nullptr;  // backing store of the StepTab arrays
  int32_t* bt = nullptr; int32_t* npages = nullptr; int32_t* free_pages = nullptr; int32_t* free_top = nullptr;
};

struct GraphKey {
  StepIO io; RuleParams rp; bool valid = false;
  bool same(const StepIO& i, const RuleParams& r) const {
    return valid && std::memcmp(&io, &i, sizeof(StepIO)) == 0 && rp.p == r.p && rp.switch_mode == r.switch_mode && rp.cap_k == r.cap_k &&
           rp.temperature == r.temperature && rp.eos_id == r.eos_id && rp.seed == r.seed && rp.top_p == r.top_p && rp.top_k == r.top_k;
  }
};

}  // namespace

struct tandem_handle {
  tandem_config cfg{};
  std::string err;
  bool cuda_fault = false;
  int esize = 4;
  int row_cap = 0, max_pages = 0, pool_pages = 0, tile_tok = 0, max_items = 0, max_comb = 0, part_cap = 0, gemm_impl = TANDEM_GEMM_SIMT, attn_impl = TANDEM_ATTN_ALU;
  int n_sms = 148;
  // tuning knobs (tandem_test_set_option; the defaults are what every measured number uses)
  int attn_ctas_per_sm = 2, gemm_ring_kb = 0;   // 0 = automatic ring size
  int gemm_pair = -1;                            // tcgen05 projections as CTA pairs (cta_group::2): -1 = automatic (while scoring: hundreds of
                                                 // rows per launch, +5%; no gain at the rollout's ~128 rows), 0 / 1 = forced
  bool scoring = false;
  bool score_nosplit = true;
  int score_chunk_grid = 8;                      // scoring: CTAs per (weight tile, K split) along the token rows (1 = off)
  bool use_pdl = true;                          // programmatic dependent launch along the kernel chain
  bool dual_forward = false;                    // measurement: the paper's lock-step engine (both models forward every token), see tandem_test.h
  bool attn_prefill_tc = true;                  // tandem_score: tcgen05 attention over 128-row q-tiles (attention_tcgen05.cuh); false = the mma.sync kernel
  bool fused_sampler = true;                    // S8 in the LM head's epilogue whenever the sampler needs no materialised logits
  int attn_min_chunk = 0;                       // 0 = by shape; "attn_min_chunk" knob for A/B
  int skip_class = -1;                          // measurement (tandem_test.h "skip_class"): the launches of this kernel class are left out of the step
  bool gateup_streamk = true;                   // gate/up + SwiGLU as the persistent stream-K kernel (gemm_streamk.cuh) when the shape allows; false = one tile per CTA
  float* sk_scratch = nullptr; int sk_rows = 0; int32_t* sk_flags = nullptr;   // its tail partials [n_sms][2][sk_rows][128] and flag / acknowledge counters [2][n_sms]
  int32_t* fault_host = nullptr; int32_t* fault_dev = nullptr;   // mapped pinned word a kernel raises when a bounded wait on another CTA expired
  size_t gemm_out_cols = 0;
  ModelWeights w[2];
  Workspace ws[2];
  StepTab tab[2]{};
  PageTab pt[2]{};
  SeqState st{};
  int32_t* st_mem = nullptr; uint8_t* st_mem8 = nullptr;
  int32_t* tokens = nullptr; uint8_t* out_owner = nullptr; float* out_logp = nullptr;
  float* score_out[2] = {nullptr, nullptr};   // tandem_score: junior log-probs and overlap [max_seqs][max_seq_len] (the senior's go to out_logp)
  float2* rope_cs = nullptr;
  uint8_t* word_start_dev = nullptr; std::vector<uint8_t> word_start_host;
  DevStats* stats = nullptr; int32_t* n_active = nullptr; int32_t* work_ctr = nullptr;
  int32_t* oom_host = nullptr; int32_t* oom_dev = nullptr;   // mapped pinned word the scheduler raises when a page pool runs dry: read by every call without a sync
  uint64_t page_order_seed = 0;                 // tandem_test_set_page_order: != 0 = pages are handed out in a seeded pseudo-random order
  cudaStream_t gs{}; cudaEvent_t ev_in{}, ev_out{};   // internal stream of the captured step graph and its fork / join events
  std::vector<uint8_t> slot_busy;           // host view of the slots
  // prompt-page sharing (cfg.share_prompt_pages): device group table and the host's view of which entries are in use
  GroupTab gt{};
  int32_t* gt_mem = nullptr; int32_t* gt_pages_mem = nullptr;
  std::vector<int> grp_free, grp_live, slot_grp;   // free group indices, members not yet seen finished per group, group of each slot
  std::vector<int> grp_reserved; int grp_released = 0;   // tandem_generate's page reservation held by each group / given back by finished groups
  // admission staging
  int32_t* stage_tokens = nullptr; size_t stage_cap = 0; long long* stage_off = nullptr; int32_t* stage_i32 = nullptr;
  // graph of one step
  cudaGraphExec_t graph = nullptr; GraphKey gkey;
  TcGemmPlans* tc = nullptr;
  CUtensorMap kv_map_store[2];
  CUtensorMap q_map_store[2];                          // each model's q buffer as [row][q-head][head_dim] in boxes of one q-tile (tcgen05 attention)
  bool q_map_ok = false;
  const CUtensorMap* kv_map[2] = {nullptr, nullptr};   // each model's whole KV pool as rows of head_dim bf16 (tensor-core attention)
  // launch accounting and the optional per-kernel-class timing mode (tandem_set_profile)
  int64_t launches = 0, graph_launches = 0, preemptions = 0;
  bool profile = false, profile_catchup_attn = false;
  std::vector<cudaEvent_t> ev_pool; size_t ev_used = 0;
  struct ProfRec { int cls; cudaEvent_t e0, e1; };
  std::vector<ProfRec> prof_pending;
  double prof_ms[TANDEM_KC_NUM] = {}; int64_t prof_n[TANDEM_KC_NUM] = {};
};

namespace {

int fail(tandem_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg;
  return code;
}
#define CU(h, expr)                                                                                  \
  do {                                                                                               \
    cudaError_t e__ = (expr);                                                                        \
    if (e__ != cudaSuccess) {                                                                        \
      (h)->cuda_fault = true;                                                                        \
      return fail((h), TANDEM_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e__));          \
    }                                                                                                \
  } while (0)

template <typename P> int dmalloc(tandem_handle* h, P** p, size_t bytes) {
  cudaError_t e = cudaMalloc((void**)p, bytes ? bytes : 16);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(h, TANDEM_ENOMEM, "cudaMalloc of " + std::to_string(bytes) + " bytes failed"); }
  return TANDEM_OK;
}
#define DM(h, p, bytes) do { int rc__ = dmalloc((h), (p), (bytes)); if (rc__) return rc__; } while (0)

// Every kernel launch of a step goes through KL: it counts the launch and, in profile mode, brackets it with a
// pair of timing events on its stream (the step then runs un-captured on one stream, see run_step).
cudaEvent_t prof_event(tandem_handle* h) {
  if (h->ev_used == h->ev_pool.size()) { cudaEvent_t e; cudaEventCreate(&e); h->ev_pool.push_back(e); }
  return h->ev_pool[h->ev_used++];
}
#define KL(h, cls, stream, ...)                                                   \
  do {                                                                            \
    if ((h)->skip_class == (cls)) break; /* measurement: this class is left out */ \
    ++(h)->launches;                                                              \
    if ((h)->profile) {                                                           \
      cudaEvent_t e0__ = prof_event(h), e1__ = prof_event(h);                     \
      cudaEventRecord(e0__, (stream));                                            \
      __VA_ARGS__;                                                                \
      cudaEventRecord(e1__, (stream));                                            \
      (h)->prof_pending.push_back({(cls), e0__, e1__});                           \
    } else {                                                                      \
      __VA_ARGS__;                                                                \
    }                                                                             \
  } while (0)

// ------------------------------------------------------------------------------------------ GEMM dispatch
// One launch for both models: out[m][s][r][n] partials (s < *n_split, stride *split_stride floats); rows of model m are
// read from rows_ptr[m] on the device.
template <typename T>
int launch_gemm(tandem_handle* h, int which, const void* const* A, const void* const* W, int N, int K, float* const* out,
                const int32_t* const* rows_ptr, int rows_cap, int* n_split, size_t* split_stride, cudaStream_t s, int epi = kTcEpiPartial,
                const TcSampleCfg* sample = nullptr) {
  const int nm = 2;
  *n_split = 1;
  *split_stride = (size_t)rows_cap * N;
  static const int cls_of[5] = {TANDEM_KC_GEMM_QKV, TANDEM_KC_GEMM_O, TANDEM_KC_GEMM_GATEUP, TANDEM_KC_GEMM_DOWN, TANDEM_KC_GEMM_LMHEAD};
  if (h->gemm_impl == TANDEM_GEMM_TCGEN05 && sizeof(T) == 2) {
    int rc = 0;
    TcGemmTune tune; tune.ring_kb = h->gemm_ring_kb; tune.pdl = h->use_pdl; tune.n_sms = h->n_sms; tune.sample = sample;
 tune.pair = h->gemm_pair >= 0 ? h->gemm_pair : (h->scoring ? 1 : 0);
    if (h->scoring && which != 4) {
      tune.chunk_grid = h->score_chunk_grid;   // hundreds of rows per launch: one CTA per 256-row chunk
      // with >= 4 chunks per weight tile the launch is wide enough without K-splits: a third of the fp32 partials to write and re-read
      if (h->score_nosplit && std::min(tune.chunk_grid, (rows_cap + kTcMaxRows - 1) / kTcMaxRows) >= 4) tune.splits = 1;
    }
    KL(h, cls_of[which], s, rc = tc_gemm_launch(h->tc, nm, which, A, W, N, K, out, rows_ptr, rows_cap, n_split, split_stride, s, epi, &tune));
    return rc == 0 ? TANDEM_OK : fail(h, rc, "tcgen05 GEMM launch failed (tensor map encode or K % 8 != 0)");
  }
  dim3 grid((N + kSimtTile - 1) / kSimtTile, std::min((rows_cap + kSimtTile - 1) / kSimtTile, 16), nm);
  Pair<SimtGemmArgs<T>> g;
  for (int m = 0; m < 2; ++m) { const int mm = m < nm ? m : 0; g.m[m] = SimtGemmArgs<T>{rows_ptr[mm], 0, (const T*)A[mm], (const T*)W[mm], out[mm], N, K}; }
  KL(h, cls_of[which], s, launch_ex(gemm_simt_kernel<T>, grid, dim3(256), 0, s, h->use_pdl, g));
  return TANDEM_OK;
}

template <typename T>
void launch_residual_norm(tandem_handle* h, cudaStream_t s, int grid_x, const Pair<ResNormArgs<T>>& a) {
  const int nm = 2;
  const int v = (a.m[0].H / 4 + 255) / 256;   // float4 per thread; tandem_init guarantees H % 8 == 0 and H <= 8192
  const dim3 grid(grid_x, nm);
  if (v <= 1) KL(h, TANDEM_KC_RESIDUAL_NORM, s, launch_ex(residual_norm_kernel<T, 256, 1>, grid, dim3(256), 0, s, h->use_pdl, a));
  else if (v <= 2) KL(h, TANDEM_KC_RESIDUAL_NORM, s, launch_ex(residual_norm_kernel<T, 256, 2>, grid, dim3(256), 0, s, h->use_pdl, a));
  else if (v <= 4) KL(h, TANDEM_KC_RESIDUAL_NORM, s, launch_ex(residual_norm_kernel<T, 256, 4>, grid, dim3(256), 0, s, h->use_pdl, a));
  else KL(h, TANDEM_KC_RESIDUAL_NORM, s, launch_ex(residual_norm_kernel<T, 256, 8>, grid, dim3(256), 0, s, h->use_pdl, a));
}

template <typename T, int D, int G>
void launch_attn_dg(const Pair<AttnArgs<T>>& a, int grid, cudaStream_t s, bool pdl) {
  launch_ex(paged_attention_kernel<T, D, G>, dim3(grid, 2), dim3(kAttnThreads), 0, s, pdl, a);
}
template <typename T> struct AttnDispatch;
template <> struct AttnDispatch<float> {
  static bool run(const Pair<AttnArgs<float>>& a, int D, int G, int grid, cudaStream_t s, bool pdl) {
#define TD_CASE(d, g) if (D == d && G == g) { launch_attn_dg<float, d, g>(a, grid, s, pdl); return true; }
    TD_CASE(32, 1) TD_CASE(32, 2) TD_CASE(32, 4) TD_CASE(64, 1) TD_CASE(64, 2) TD_CASE(64, 4) TD_CASE(128, 1) TD_CASE(128, 2) TD_CASE(128, 4)
#undef TD_CASE
    return false;
  }
};
template <> struct AttnDispatch<bf16> {
  static bool run(const Pair<AttnArgs<bf16>>& a, int D, int G, int grid, cudaStream_t s, bool pdl) {
#define TD_CASE(d, g) if (D == d && G == g) { launch_attn_dg<bf16, d, g>(a, grid, s, pdl); return true; }
    TD_CASE(64, 1) TD_CASE(64, 2) TD_CASE(64, 4) TD_CASE(64, 7) TD_CASE(64, 8) TD_CASE(128, 1) TD_CASE(128, 2) TD_CASE(128, 4) TD_CASE(128, 8)
#undef TD_CASE
    return false;
  }
};
template <int D, int G> struct AmStages { static constexpr int value = D == 128 ? 2 : 4; };
template <int D, int G>
bool launch_attn_mma_dg(const Pair<CUtensorMap>& map, const Pair<AttnMmaArgs>& a, int grid, cudaStream_t s, bool set_attr, bool pdl) {
  constexpr int ST = AmStages<D, G>::value;
  constexpr int smem = attn_mma_smem_bytes<D, ST>();
  if (set_attr) return cudaFuncSetAttribute(paged_attention_mma_kernel<D, G, ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) == cudaSuccess;
  return launch_ex(paged_attention_mma_kernel<D, G, ST>, dim3(grid), dim3(kAmThreads), smem, s, pdl, map, a) == cudaSuccess;
}
// set_attr = true: only raise the kernel's dynamic shared memory limit (called once from tandem_init)
bool run_attn_mma(const Pair<CUtensorMap>& map, const Pair<AttnMmaArgs>& a, int D, int G, int grid, cudaStream_t s, bool set_attr, bool pdl = false) {
#define TD_CASE(d, g) if (D == d && G == g) return launch_attn_mma_dg<d, g>(map, a, grid, s, set_attr, pdl);
  TD_CASE(64, 1) TD_CASE(64, 2) TD_CASE(64, 4) TD_CASE(64, 7) TD_CASE(64, 8) TD_CASE(128, 1) TD_CASE(128, 2) TD_CASE(128, 4) TD_CASE(128, 8)
#undef TD_CASE
  return false;
}
// tcgen05 attention for scoring (attention_tcgen05.cuh): set_attr = true raises the dynamic shared memory limit only
bool run_attn_tc(const Pair<CUtensorMap>& kv, const Pair<CUtensorMap>& q, const Pair<AttnMmaArgs>& a, int D, int G, int grid, cudaStream_t s, bool set_attr, bool pdl = false) {
  if (D == 128) {
    if (set_attr) return cudaFuncSetAttribute(prefill_attention_tc_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_tc_smem_bytes<128>()) == cudaSuccess;
    return launch_ex(prefill_attention_tc_kernel<128>, dim3(grid), dim3(kAtThreads), attn_tc_smem_bytes<128>(), s, pdl, kv, q, a, G) == cudaSuccess;
  }
  if (D == 64) {
    if (set_attr) return cudaFuncSetAttribute(prefill_attention_tc_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_tc_smem_bytes<64>()) == cudaSuccess;
    return launch_ex(prefill_attention_tc_kernel<64>, dim3(grid), dim3(kAtThreads), attn_tc_smem_bytes<64>(), s, pdl, kv, q, a, G) == cudaSuccess;
  }
  return false;
}
bool use_attn_tc(const tandem_handle* h) { return h->attn_prefill_tc && h->attn_impl == TANDEM_ATTN_MMA && h->q_map_ok; }
bool attn_supported(int dtype, int D, int G) {
  if (dtype == TANDEM_F32) return (D == 32 || D == 64 || D == 128) && (G == 1 || G == 2 || G == 4);
  return (D == 64 && (G == 1 || G == 2 || G == 4 || G == 7 || G == 8)) || (D == 128 && (G == 1 || G == 2 || G == 4 || G == 8));
}

// ------------------------------------------------------------------------------------------ both models' forward (S1..S8)
// Every kernel is launched once for the two models (Pair arguments): the models advance layer by layer in lock-step on
// one stream, each launch carrying the senior's and the junior's half of the work.
template <typename T>
int forward_pair(tandem_handle* h, const StepIO& io, const RuleParams& rp, cudaStream_t s, bool score = false, float score_inv_t = 1.f) {
  const tandem_config& c = h->cfg;
  const int H = c.hidden, nq = c.n_q_heads, nkv = c.n_kv_heads, d = c.head_dim, I = c.intermediate, V = c.vocab;
  const int qkv_n = (nq + 2 * nkv) * d;
  const int row_grid = h->n_sms * 2;
  const size_t layer_kv = (size_t)2 * h->pool_pages * nkv * kPageTokens * d;
  const size_t half_kv = (size_t)h->pool_pages * nkv * kPageTokens * d;
  const bool mma = h->attn_impl == TANDEM_ATTN_MMA;
  const bool pdl = h->use_pdl;
  int ns; size_t ss; int rc;
  const void* A[2]; const void* W[2]; float* O[2]; const int32_t* RP[2];
  auto set_gemm = [&](int m, const void* a_, const void* w_, float* o_, const int32_t* r_) { A[m] = a_; W[m] = w_; O[m] = o_; RP[m] = r_; };

  {
    Pair<EmbedArgs<T>> ea;
    for (int m = 0; m < 2; ++m) ea.m[m] = EmbedArgs<T>{h->tab[m].counts, h->tab[m].row_tok, (const T*)h->w[m].embed, (const T*)h->w[m].attn_norm[0], h->ws[m].x, (T*)h->ws[m].act, H, c.rms_eps};
    KL(h, TANDEM_KC_EMBED, s, launch_ex(embed_norm_kernel<T, 256>, dim3(row_grid, 2), dim3(256), 0, s, false, ea));
  }

  for (int l = 0; l < c.n_layers; ++l) {
    // S3 QKV projection
    for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].act, h->w[m].wqkv[l], h->ws[m].gemm_out, h->tab[m].counts + C_ROWS);
    if ((rc = launch_gemm<T>(h, 0, A, W, qkv_n, H, O, RP, h->row_cap, &ns, &ss, s))) return rc;
    // S4 RoPE + KV append
    if (mma) {
      Pair<RopeArgs<T, bf16>> ra;
      for (int m = 0; m < 2; ++m) {
        T* kpool = (T*)h->ws[m].kv + (size_t)l * layer_kv;
        ra.m[m] = RopeArgs<T, bf16>{h->tab[m].counts, h->tab[m].row_pos, h->tab[m].row_kvslot, h->ws[m].gemm_out, ns, ss, h->rope_cs, (bf16*)h->ws[m].q, kpool, kpool + half_kv, nq, nkv, d};
      }
      KL(h, TANDEM_KC_ROPE_APPEND, s, launch_ex(rope_append_kernel<T, bf16, 256>, dim3(row_grid * 4, 2), dim3(256), 0, s, pdl, ra));
    } else {
      Pair<RopeArgs<T, float>> ra;
      for (int m = 0; m < 2; ++m) {
        T* kpool = (T*)h->ws[m].kv + (size_t)l * layer_kv;
        ra.m[m] = RopeArgs<T, float>{h->tab[m].counts, h->tab[m].row_pos, h->tab[m].row_kvslot, h->ws[m].gemm_out, ns, ss, h->rope_cs, (float*)h->ws[m].q, kpool, kpool + half_kv, nq, nkv, d};
      }
      KL(h, TANDEM_KC_ROPE_APPEND, s, launch_ex(rope_append_kernel<T, float, 256>, dim3(row_grid * 4, 2), dim3(256), 0, s, pdl, ra));
    }
    // S5 attention (decode splits + catch-up rows)
    {
      bool ok = true;
      if (mma) {
        const long long rows_per_half = (long long)h->pool_pages * nkv * kPageTokens;
        Pair<AttnMmaArgs> ma; Pair<CUtensorMap> maps;
        for (int m = 0; m < 2; ++m) {
          const StepTab& tb = h->tab[m];
          ma.m[m] = AttnMmaArgs{tb.counts, tb.item_row0, tb.item_ntok, tb.item_kv0, tb.item_kv1, tb.item_part, tb.row_slot, tb.row_pos, h->pt[m].bt, h->max_pages,
                                (const bf16*)h->ws[m].q, (bf16*)h->ws[m].attn_out, h->ws[m].part_acc, h->ws[m].part_ml, nq, nkv, 1.0f / sqrtf((float)d),
                                (int)((2ll * l) * rows_per_half), (int)((2ll * l + 1) * rows_per_half), h->work_ctr + l, 0};
          maps.m[m] = h->kv_map_store[m];
        }
        if (score && use_attn_tc(h)) {
          Pair<CUtensorMap> qm; qm.m[0] = h->q_map_store[0]; qm.m[1] = h->q_map_store[1];
          KL(h, TANDEM_KC_ATTENTION, s, ok = run_attn_tc(maps, qm, ma, d, nq / nkv, 2 * h->n_sms, s, false, pdl));
        } else
        KL(h, TANDEM_KC_ATTENTION, s, ok = run_attn_mma(maps, ma, d, nq / nkv, h->attn_ctas_per_sm * h->n_sms, s, false, pdl));
        if (ok && h->profile && h->profile_catchup_attn) {
          // measurement (BASELINE.json configs[4], "catch-up-prefill share of step time"): the same launch again, restricted to the items
          // with more than one query token (S5b); it rewrites the same values, so results are unchanged
          for (int m = 0; m < 2; ++m) { ma.m[m].min_ntok = 2; ma.m[m].work_ctr = h->work_ctr + c.n_layers + l; }
          KL(h, TANDEM_KC_ATTN_CATCHUP, s, ok = run_attn_mma(maps, ma, d, nq / nkv, h->attn_ctas_per_sm * h->n_sms, s, false, pdl));
          // and once more with every item filtered out: the fixed cost of such a launch, to be subtracted
          for (int m = 0; m < 2; ++m) { ma.m[m].min_ntok = 1 << 30; ma.m[m].work_ctr = h->work_ctr + 2 * c.n_layers + l; }
          KL(h, TANDEM_KC_ATTN_EMPTY, s, ok = ok && run_attn_mma(maps, ma, d, nq / nkv, h->attn_ctas_per_sm * h->n_sms, s, false, pdl));
        }
      } else {
        Pair<AttnArgs<T>> aa;
        for (int m = 0; m < 2; ++m) {
          const StepTab& tb = h->tab[m];
          T* kpool = (T*)h->ws[m].kv + (size_t)l * layer_kv;
          aa.m[m] = AttnArgs<T>{tb.counts, tb.item_row0, tb.item_ntok, tb.item_kv0, tb.item_kv1, tb.item_part, tb.row_slot, tb.row_pos, h->pt[m].bt, h->max_pages,
                                (const float*)h->ws[m].q, kpool, kpool + half_kv, (T*)h->ws[m].attn_out, h->ws[m].part_acc, h->ws[m].part_ml, nq, nkv, 1.0f / sqrtf((float)d)};
        }
        KL(h, TANDEM_KC_ATTENTION, s, ok = AttnDispatch<T>::run(aa, d, nq / nkv, h->n_sms * 2, s, pdl));
      }
      if (!ok) return fail(h, TANDEM_EINVAL, "unsupported (head_dim, group) for attention");
    }
    {
      Pair<CombineArgs<T>> ca;
      for (int m = 0; m < 2; ++m) {
        const StepTab& tb = h->tab[m];
        ca.m[m] = CombineArgs<T>{tb.counts, tb.comb_row, tb.comb_part0, tb.comb_n, tb.comb_stride, tb.comb_gpart, h->ws[m].part_acc, h->ws[m].part_ml, (T*)h->ws[m].attn_out, nq, d};
      }
      KL(h, TANDEM_KC_ATTN_COMBINE, s, launch_ex(attn_combine_kernel<T>, dim3(h->n_sms * 4, 2), dim3(256), 0, s, pdl, ca));
    }
    // S6 O projection + residual + RMSNorm(mlp)
    for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].attn_out, h->w[m].wo[l], h->ws[m].gemm_out, h->tab[m].counts + C_ROWS);
    if ((rc = launch_gemm<T>(h, 1, A, W, H, nq * d, O, RP, h->row_cap, &ns, &ss, s))) return rc;
    {
      Pair<ResNormArgs<T>> na;
      for (int m = 0; m < 2; ++m)
        na.m[m] = ResNormArgs<T>{h->tab[m].counts, h->ws[m].gemm_out, ns, ss, h->ws[m].x, (const T*)h->w[m].mlp_norm[l], (T*)h->ws[m].act, nullptr, H, c.rms_eps};
      launch_residual_norm<T>(h, s, row_grid, na);
    }
    // S7 gate/up + SwiGLU, down + residual + RMSNorm(next layer | final)
    if (h->gemm_impl == TANDEM_GEMM_TCGEN05) {   // SwiGLU in the GEMM epilogue (gate/up rows interleaved at load time)
      for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].act, h->w[m].wgu[l], (float*)h->ws[m].mlp_act, h->tab[m].counts + C_ROWS);
      if (h->sk_scratch && h->gateup_streamk && !h->scoring) {   // decode-sized steps: stream-K over tile pairs, both models, one CTA per SM
        void* outs[2] = {h->ws[0].mlp_act, h->ws[1].mlp_act};
        int src = 0;
        KL(h, TANDEM_KC_GEMM_GATEUP, s, src = sk_gateup_launch(h->tc, A, W, 2 * I, H, outs, RP, h->row_cap, h->sk_scratch, h->sk_rows, h->sk_flags,
                                                              h->sk_flags + h->n_sms, h->fault_dev, h->n_sms, s, pdl));
        if (src) return fail(h, src, "stream-K gate/up launch failed");
      } else if ((rc = launch_gemm<T>(h, 2, A, W, 2 * I, H, O, RP, h->row_cap, &ns, &ss, s, kTcEpiSwiGLU))) return rc;
    } else {
      for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].act, h->w[m].wgu[l], h->ws[m].gemm_out, h->tab[m].counts + C_ROWS);
      if ((rc = launch_gemm<T>(h, 2, A, W, 2 * I, H, O, RP, h->row_cap, &ns, &ss, s))) return rc;
      Pair<SwigluArgs<T>> sg;
      for (int m = 0; m < 2; ++m) sg.m[m] = SwigluArgs<T>{h->tab[m].counts, h->ws[m].gemm_out, ns, ss, (T*)h->ws[m].mlp_act, I};
      KL(h, TANDEM_KC_SWIGLU, s, launch_ex(swiglu_kernel<T, 256>, dim3(row_grid, 2), dim3(256), 0, s, pdl, sg));
    }
    for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].mlp_act, h->w[m].wdown[l], h->ws[m].gemm_out, h->tab[m].counts + C_ROWS);
    if ((rc = launch_gemm<T>(h, 3, A, W, H, I, O, RP, h->row_cap, &ns, &ss, s))) return rc;
    const bool last = l == c.n_layers - 1;
    {
      Pair<ResNormArgs<T>> na;
      for (int m = 0; m < 2; ++m)
        na.m[m] = ResNormArgs<T>{h->tab[m].counts, h->ws[m].gemm_out, ns, ss, h->ws[m].x, (const T*)(last ? h->w[m].final_norm : h->w[m].attn_norm[l + 1]),
                                 (T*)(last ? (score ? h->ws[m].score_lm_in : h->ws[m].lm_in) : h->ws[m].act), last ? h->tab[m].row_emit : nullptr, H, c.rms_eps};
      launch_residual_norm<T>(h, s, row_grid, na);
    }
  }
  if (score) {   // every row reaches the LM head (the scheduler set row_emit[r] = r); the dual-scoring kernel replaces the sampler
    for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].score_lm_in, h->w[m].lm_head, h->ws[m].score_logits, h->tab[m].counts + C_EMIT);
    if ((rc = launch_gemm<T>(h, 4, A, W, V, H, O, RP, h->row_cap, &ns, &ss, s))) return rc;
    const ScoreArgs sc{h->tab[0].counts, h->tab[0].row_slot, h->tab[0].row_pos, h->tokens, c.max_seq_len, h->ws[0].score_logits, h->ws[1].score_logits, V,
                       score_inv_t, h->out_logp, h->score_out[0], h->score_out[1]};
    KL(h, TANDEM_KC_SCORE, s, launch_ex(score_kernel<512>, dim3(h->row_cap), dim3(512), 0, s, pdl, sc));
    return TANDEM_OK;
  }
  // S8 LM head on the emitting rows only, then sample + switch + emit
  const bool want_nucleus = rp.temperature > 0.f && (rp.top_p < 1.f || (rp.top_k > 0 && rp.top_k < V));
  if (h->fused_sampler && h->gemm_impl == TANDEM_GEMM_TCGEN05 && sizeof(T) == 2 && !want_nucleus && !io.u_sample && !io.dbg_logits && !io.forced_tokens) {
    // the default sampling path: (max, sum exp, argmax, Gumbel-max) are reduced in the LM head's epilogue per 128-id weight tile and merged
    // by one warp per row - no [rows, V] logits in HBM. Filters, explicit uniforms, forced tokens and the logits tap need the logits.
    const bool greedy = !(rp.temperature > 0.f);
    const TcSampleCfg sc{{h->tab[0].emit_slot, h->tab[1].emit_slot}, h->st.n_emit, h->st.seq_id, greedy ? 1.f : 1.f / rp.temperature, greedy ? 1 : 0, rp.seed};
    for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].lm_in, h->w[m].lm_head, h->ws[m].spart, h->tab[m].counts + C_EMIT);
    if ((rc = launch_gemm<T>(h, 4, A, W, V, H, O, RP, c.max_seqs, &ns, &ss, s, kTcEpiSample, &sc))) return rc;
    Pair<SampleMergeArgs> sm;
    for (int m = 0; m < 2; ++m)
      sm.m[m] = SampleMergeArgs{SampleArgs{h->st, h->tab[m], io, rp, nullptr, h->word_start_dev, h->tokens, h->out_owner, h->out_logp, V, c.max_seq_len, m, nullptr, nullptr, 0},
                                h->ws[m].spart, (V + kTcTileN - 1) / kTcTileN, c.max_seqs};
    KL(h, TANDEM_KC_SAMPLE, s, launch_ex(sample_merge_emit_kernel<128>, dim3((c.max_seqs + 3) / 4, 2), dim3(128), 0, s, pdl, sm));
    return TANDEM_OK;
  }
  for (int m = 0; m < 2; ++m) set_gemm(m, h->ws[m].lm_in, h->w[m].lm_head, h->ws[m].logits, h->tab[m].counts + C_EMIT);
  if ((rc = launch_gemm<T>(h, 4, A, W, V, H, O, RP, c.max_seqs, &ns, &ss, s))) return rc;
  Pair<SampleArgs> sa;
  const int n_chunk = std::max(1, std::min(kSampleMaxChunks, V / 8192));   // ~8k ids per CTA: 18 slices at V = 151,936
  for (int m = 0; m < 2; ++m)
    sa.m[m] = SampleArgs{h->st, h->tab[m], io, rp, h->ws[m].logits, h->word_start_dev, h->tokens, h->out_owner, h->out_logp, V, c.max_seq_len, m,
                         h->ws[m].chunk_part, h->ws[m].chunk_ctr, n_chunk};
  const size_t nucleus_smem = want_nucleus ? sizeof(NucleusSmem<256>) : 0;
  if (nucleus_smem) KL(h, TANDEM_KC_SAMPLE, s, launch_ex(sample_switch_emit_kernel<256, true>, dim3(c.max_seqs, n_chunk, 2), dim3(256), nucleus_smem, s, pdl, sa));
  else KL(h, TANDEM_KC_SAMPLE, s, launch_ex(sample_switch_emit_kernel<256, false>, dim3(c.max_seqs, n_chunk, 2), dim3(256), 0, s, pdl, sa));
  return TANDEM_OK;
}

int launch_step(tandem_handle* h, const StepIO& io, const RuleParams& rp, cudaStream_t s, bool score = false, float score_inv_t = 1.f) {
  const tandem_config& c = h->cfg;
  SchedArgs sa{};
  sa.st = h->st; sa.pt[0] = h->pt[0]; sa.pt[1] = h->pt[1]; sa.gt = h->gt; sa.tab[0] = h->tab[0]; sa.tab[1] = h->tab[1];
  sa.io = io; sa.stats = h->stats; sa.tokens = h->tokens; sa.max_seqs = c.max_seqs; sa.max_seq_len = c.max_seq_len;
  sa.max_pages = h->max_pages; sa.row_cap = h->row_cap; sa.tile_tok = h->tile_tok;
  if (score && use_attn_tc(h)) { sa.tile_tok = kAtTileKv / (c.n_q_heads / c.n_kv_heads); sa.no_parts = 1; }   // 128-row q-tiles, each over its whole causal range
  sa.work_ctr = h->work_ctr; sa.n_work_ctr = 3 * c.n_layers;
  sa.cascade = (c.share_prompt_pages == 2 && !score) ? 1 : 0;
  sa.min_chunk = h->attn_min_chunk > 0 ? h->attn_min_chunk : (c.n_kv_heads >= 8 ? kAttnMinChunkWide : kAttnMinChunk);
  sa.score = score ? 1 : 0; sa.oom_flag = h->oom_dev; sa.lockstep = (h->dual_forward && !score) ? 1 : 0;
  KL(h, TANDEM_KC_SCHED, s, (sched_kernel<<<1, 1024, 0, s>>>(sa)));
  const int rc = (c.dtype == TANDEM_F32) ? forward_pair<float>(h, io, rp, s, score, score_inv_t) : forward_pair<bf16>(h, io, rp, s, score, score_inv_t);
  if (rc) return rc;
  FinalArgs fa{h->st, {h->pt[0], h->pt[1]}, h->gt, io, h->stats, h->n_active, c.max_seqs, h->max_pages, h->pool_pages};
  KL(h, TANDEM_KC_FINALIZE, s, (finalize_kernel<<<1, 1024, 0, s>>>(fa)));
  return TANDEM_OK;
}

// One step, through the captured graph when enabled and the (io, rule) key is unchanged.
int run_step(tandem_handle* h, const StepIO& io, const RuleParams& rp, cudaStream_t s) {
  if (h->profile) {
    h->ev_used = 0; h->prof_pending.clear();
    const int rc = launch_step(h, io, rp, s);
    if (rc) return rc;
    CU(h, cudaStreamSynchronize(s));
    for (const auto& r : h->prof_pending) {
      float ms = 0.f;
      CU(h, cudaEventElapsedTime(&ms, r.e0, r.e1));
      h->prof_ms[r.cls] += ms; h->prof_n[r.cls] += 1;
    }
    return TANDEM_OK;
  }
  if (!h->cfg.use_graph) {
    const int rc = launch_step(h, io, rp, s);
    if (rc) return rc;
    CU(h, cudaGetLastError());
    return TANDEM_OK;
  }
  // the graph lives on an internal stream (the caller's may be the legacy default stream, which cannot capture)
  if (!h->gkey.same(io, rp)) {
    if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }
    h->gkey.valid = false;
    cudaGraph_t g = nullptr;
    const int64_t l0 = h->launches;
    CU(h, cudaStreamBeginCapture(h->gs, cudaStreamCaptureModeThreadLocal));
    const int rc = launch_step(h, io, rp, h->gs);
    cudaError_t e = cudaStreamEndCapture(h->gs, &g);
    if (rc) { if (g) cudaGraphDestroy(g); return rc; }
    CU(h, e);
    CU(h, cudaGraphInstantiate(&h->graph, g, 0));
    cudaGraphDestroy(g);
    h->gkey.io = io; h->gkey.rp = rp; h->gkey.valid = true;
    h->graph_launches = h->launches - l0;
    h->launches = l0;   // capturing launched nothing
  }
  h->launches += h->graph_launches;
  CU(h, cudaEventRecord(h->ev_in, s));
  CU(h, cudaStreamWaitEvent(h->gs, h->ev_in, 0));
  CU(h, cudaGraphLaunch(h->graph, h->gs));
  CU(h, cudaEventRecord(h->ev_out, h->gs));
  CU(h, cudaStreamWaitEvent(s, h->ev_out, 0));
  return TANDEM_OK;
}

int check_params(tandem_handle* h, const tandem_params* p) {
  if (!p) return fail(h, TANDEM_EINVAL, "params is NULL");
  if (!(p->p >= 0.f && p->p <= 1.f)) return fail(h, TANDEM_EINVAL, "p must be in [0,1]");
  if (p->switch_mode != TANDEM_TOGGLE && p->switch_mode != TANDEM_REDRAW) return fail(h, TANDEM_EINVAL, "bad switch_mode");
  if (p->start_owner < 0 || p->start_owner > 2) return fail(h, TANDEM_EINVAL, "bad start_owner");
  if (p->cap_k < 0) return fail(h, TANDEM_EINVAL, "cap_k must be >= 0");
  if (!(p->temperature >= 0.f)) return fail(h, TANDEM_EINVAL, "temperature must be >= 0");
  if (!(p->top_p > 0.f && p->top_p <= 1.0f)) return fail(h, TANDEM_EINVAL, "top_p must be in (0, 1]");
  if (p->top_k > kNucleusCap && p->top_k < h->cfg.vocab) return fail(h, TANDEM_EINVAL, "top_k above 2048 (and below vocab) is not supported");
  if (p->eos_id >= h->cfg.vocab) return fail(h, TANDEM_EINVAL, "eos_id >= vocab");
  if (!p->word_start) return fail(h, TANDEM_EINVAL, "word_start is NULL");
  return TANDEM_OK;
}

int sync_word_start(tandem_handle* h, const tandem_params* p, cudaStream_t s) {
  const size_t V = (size_t)h->cfg.vocab;
  if (h->word_start_host.size() == V && std::memcmp(h->word_start_host.data(), p->word_start, V) == 0) return TANDEM_OK;
  h->word_start_host.assign(p->word_start, p->word_start + V);
  CU(h, cudaStreamSynchronize(s));
  CU(h, cudaMemcpy(h->word_start_dev, h->word_start_host.data(), V, cudaMemcpyHostToDevice));
  return TANDEM_OK;
}

StepIO make_io(const tandem_step_out* out, const tandem_overrides* ovr) {
  StepIO io{};
  if (out) { io.token = out->token; io.owner = out->owner; io.sen_logp = out->sen_logp; io.done = out->done; io.argmax = out->argmax; io.n_active = out->n_active; }
  if (ovr) {
    io.forced_tokens = ovr->forced_tokens; io.forced_stride = ovr->forced_stride;
    io.u_switch = ovr->u_switch; io.u_switch_stride = ovr->u_switch_stride;
    io.u_sample = ovr->u_sample; io.u_sample_stride = ovr->u_sample_stride;
    io.dbg_logits = ovr->dbg_logits;
  }
  return io;
}
RuleParams make_rule(const tandem_params* p) {
  RuleParams r{}; r.p = p->p; r.switch_mode = p->switch_mode; r.cap_k = p->cap_k; r.temperature = p->temperature; r.eos_id = p->eos_id; r.seed = p->seed; r.top_p = p->top_p; r.top_k = p->top_k;
  return r;
}

// Refresh the host view of the slots (a slot is free once the finalize kernel cleared its active flag).
int refresh_slots(tandem_handle* h, cudaStream_t s) {
  std::vector<uint8_t> act(h->cfg.max_seqs);
  CU(h, cudaStreamSynchronize(s));
  CU(h, cudaMemcpy(act.data(), h->st.active, act.size(), cudaMemcpyDeviceToHost));
  for (int i = 0; i < h->cfg.max_seqs; ++i) {
    if (h->slot_busy[i] && !act[i] && h->slot_grp[i] >= 0) {   // a member finished: the group's index is reusable after its last one
      const int g = h->slot_grp[i];
      if (--h->grp_live[g] == 0) { h->grp_free.push_back(g); h->grp_released += h->grp_reserved[g]; h->grp_reserved[g] = 0; }
      h->slot_grp[i] = -1;
    }
    h->slot_busy[i] = act[i];
  }
  return TANDEM_OK;
}

int admit(tandem_handle* h, const tandem_params* p, const tandem_overrides* ovr, int n, const int32_t* toks, const int64_t* offs,
          const int32_t* seq_ids, const int32_t* max_new, int32_t* slots_out, cudaStream_t s, bool score = false) {
  const tandem_config& c = h->cfg;
  if (n <= 0) return TANDEM_OK;
  if (!toks || !offs || !max_new) return fail(h, TANDEM_EINVAL, "admission arrays are NULL");
  std::vector<int32_t> slots;
  for (int i = 0; i < c.max_seqs && (int)slots.size() < n; ++i) if (!h->slot_busy[i]) slots.push_back(i);
  if ((int)slots.size() < n) return fail(h, TANDEM_EFULL, "not enough free slots");
  const int64_t total = offs[n] - offs[0];
  for (int i = 0; i < n; ++i) {
    const int64_t len = offs[i + 1] - offs[i];
    if (len < 1) return fail(h, TANDEM_EINVAL, "empty prompt");
    if (max_new[i] < 1) return fail(h, TANDEM_EINVAL, "max_new must be >= 1");
    if (len + (score ? 0 : max_new[i]) > c.max_seq_len) return fail(h, TANDEM_EINVAL, score ? "stream longer than max_seq_len" : "prompt + max_new exceeds max_seq_len");
  }
  for (int64_t k = offs[0]; k < offs[n]; ++k) if (toks[k] < 0 || toks[k] >= c.vocab) return fail(h, TANDEM_EINVAL, "token id out of range");
  if ((size_t)total > h->stage_cap) {
    if (h->stage_tokens) cudaFree(h->stage_tokens);
    h->stage_tokens = nullptr; h->stage_cap = 0;
    DM(h, &h->stage_tokens, (size_t)total * 4);
    h->stage_cap = (size_t)total;
  }
  std::vector<long long> o(n + 1);
  std::vector<int32_t> meta(5 * (size_t)n);
  for (int i = 0; i <= n; ++i) o[i] = offs[i] - offs[0];
  for (int i = 0; i < n; ++i) { meta[i] = slots[i]; meta[n + i] = seq_ids ? seq_ids[i] : slots[i]; meta[2 * n + i] = max_new[i]; meta[3 * n + i] = -1; meta[4 * n + i] = 0; }
  if (c.share_prompt_pages && !score) {
    // Groups = runs of consecutive sequences of this call with identical prompts of more than one page (the G rollouts of a
    // prompt): they share the full pages of the prompt except the one holding its last token.
    for (int i = 0; i < n;) {
      const int64_t len = offs[i + 1] - offs[i];
      int j = i + 1;
      while (j < n && offs[j + 1] - offs[j] == len && std::memcmp(toks + offs[i], toks + offs[j], (size_t)len * 4) == 0) ++j;
      if (j - i >= 2 && (len - 1) / kPageTokens >= 1 && !h->grp_free.empty()) {
        const int g = h->grp_free.back(); h->grp_free.pop_back();
        h->grp_live[g] = j - i;
        for (int k = i; k < j; ++k) { meta[3 * n + k] = g; h->slot_grp[slots[k]] = g; }
        meta[4 * n + i] = j - i;
      }
      i = j;
    }
  }
  CU(h, cudaStreamSynchronize(s));
  CU(h, cudaMemcpy(h->stage_tokens, toks + offs[0], (size_t)total * 4, cudaMemcpyHostToDevice));
  CU(h, cudaMemcpy(h->stage_off, o.data(), (n + 1) * sizeof(long long), cudaMemcpyHostToDevice));
  CU(h, cudaMemcpy(h->stage_i32, meta.data(), meta.size() * 4, cudaMemcpyHostToDevice));
  AdmitArgs a{};
  a.st = h->st; a.pt[0] = h->pt[0]; a.pt[1] = h->pt[1]; a.gt = h->gt; a.tokens = h->tokens; a.max_seq_len = c.max_seq_len;
  a.stage_tokens = h->stage_tokens; a.stage_off = h->stage_off; a.slots = h->stage_i32; a.seq_ids = h->stage_i32 + n; a.max_new = h->stage_i32 + 2 * n;
  a.grp = h->stage_i32 + 3 * n; a.grp_members = h->stage_i32 + 4 * n;
  a.n = n; a.start_owner = p->start_owner; a.p = p->p; a.seed = p->seed;
  a.u_switch = ovr ? ovr->u_switch : nullptr; a.u_switch_stride = ovr ? ovr->u_switch_stride : 0;
  admit_kernel<<<n, 128, 0, s>>>(a);
  CU(h, cudaGetLastError());
  CU(h, cudaStreamSynchronize(s));
  for (int i = 0; i < n; ++i) { h->slot_busy[slots[i]] = 1; if (slots_out) slots_out[i] = slots[i]; }
  return TANDEM_OK;
}

int fill_stats(tandem_handle* h, tandem_stats* stats) {
  const tandem_config& c = h->cfg;
  DevStats d;
  CU(h, cudaMemcpy(&d, h->stats, sizeof(d), cudaMemcpyDeviceToHost));
  const int H = c.hidden, I = c.intermediate, qd = c.n_q_heads * c.head_dim, kd = c.n_kv_heads * c.head_dim;
  const int64_t per_layer = (int64_t)H * qd + 2ll * H * kd + (int64_t)qd * H + 3ll * H * I + 2ll * H;
  const int64_t wbytes = ((int64_t)c.n_layers * per_layer + H + (int64_t)c.vocab * H) * h->esize;
  stats->steps = (int64_t)d.steps; stats->tokens_emitted = (int64_t)d.tokens_emitted;
  stats->rows_senior = (int64_t)d.rows[0]; stats->rows_junior = (int64_t)d.rows[1]; stats->catchup_rows = (int64_t)d.catchup_rows;
  stats->kv_bytes_read = (int64_t)d.kv_tokens_read * 2ll * c.n_layers * kd * h->esize;
  stats->weight_bytes_read = (int64_t)d.model_steps * wbytes;
  stats->peak_pages_senior = d.peak_pages_used[0]; stats->peak_pages_junior = d.peak_pages_used[1]; stats->peak_resident = d.peak_resident;
  stats->seconds_total = 0.0;
  stats->kernel_launches = h->launches;
  stats->shared_prompt_rows = (int64_t)d.shared_rows;
  stats->kv_bytes_shared_reads = (int64_t)d.kv_tokens_shared * 2ll * c.n_layers * kd * h->esize;
  stats->starved = (int64_t)d.starved; stats->preemptions = h->preemptions;
  return TANDEM_OK;
}

int check_ready(tandem_handle* h) {
  if (!h) return TANDEM_EINVAL;
  if (h->cuda_fault) return fail(h, TANDEM_ECUDA, "a previous CUDA error is sticky: " + h->err);
  if (!h->w[0].loaded || !h->w[1].loaded) return fail(h, TANDEM_ESTATE, "weights of both models must be loaded first");
  return TANDEM_OK;
}

struct EventPair {   // timing events of tandem_generate / tandem_score, destroyed on every exit path
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  ~EventPair() { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); }
};

// KV-pool exhaustion seen by the scheduler of an earlier step (mapped host word, no synchronisation): sticky until tandem_reset
int check_oom_flag(tandem_handle* h) {
  if (h->fault_host && *(volatile int32_t*)h->fault_host)
    return fail(h, TANDEM_ECUDA, "a kernel's bounded wait on another CTA expired (stream-K hand-over): results since then are invalid; tandem_free the handle");
  if (h->oom_host && *(volatile int32_t*)h->oom_host >= 2)
    return fail(h, TANDEM_ENOMEM, "KV page pools exhausted: every resident sequence is stalled and no step can make progress (nothing was corrupted); "
                                  "tandem_reset the handle, then enlarge kv_bytes_per_model or admit fewer sequences");
  return TANDEM_OK;
}

int check_oom(tandem_handle* h, cudaStream_t s) {
  DevStats st;
  CU(h, cudaStreamSynchronize(s));
  CU(h, cudaMemcpy(&st, h->stats, sizeof(st), cudaMemcpyDeviceToHost));
  if (h->oom_host && *(volatile int32_t*)h->oom_host >= 2) return check_oom_flag(h);
  (void)st;
  return TANDEM_OK;
}

// Preemption: the sequence in `slot` gives its pages back (its own ones at once, its group's shared prompt pages with the group's last
// member) and the slot becomes free - the finalize kernel's path for a finished sequence, taken early.
int preempt_slot(tandem_handle* h, int slot, cudaStream_t s) {
  const tandem_config& c = h->cfg;
  const uint8_t one = 1;
  CU(h, cudaMemcpyAsync(h->st.done + slot, &one, 1, cudaMemcpyHostToDevice, s));
  FinalArgs fa{h->st, {h->pt[0], h->pt[1]}, h->gt, StepIO{}, h->stats, h->n_active, c.max_seqs, h->max_pages, h->pool_pages};
  finalize_kernel<<<1, 1024, 0, s>>>(fa);
  CU(h, cudaGetLastError());
  return refresh_slots(h, s);
}

}  // namespace

// =================================================================================================== C ABI
extern "C" {

int tandem_init(const tandem_config* cfg, tandem_handle** out) {
  if (!cfg || !out) return TANDEM_EINVAL;
  *out = nullptr;
  tandem_handle* h = new tandem_handle();
  h->cfg = *cfg;
  const tandem_config& c = h->cfg;
  auto bad = [&](const char* m) { int rc = fail(h, TANDEM_EINVAL, m); fprintf(stderr, "tandem_init: %s\n", m); tandem_free(h); return rc; };   // frees whatever was allocated so far
  if (c.n_layers < 1 || c.hidden < 8 || c.n_q_heads < 1 || c.n_kv_heads < 1 || c.head_dim < 8 || c.intermediate < 8 || c.vocab < 2) return bad("bad model dimensions");
  if (c.n_q_heads % c.n_kv_heads) return bad("n_q_heads must be a multiple of n_kv_heads");
  if ((c.hidden % 8) || (c.intermediate % 8) || (c.head_dim % 8) || c.hidden > 8192) return bad("hidden, intermediate, head_dim must be multiples of 8; hidden <= 8192");
  if (c.dtype != TANDEM_F32 && c.dtype != TANDEM_BF16) return bad("bad dtype");
  if (c.page_tokens != kPageTokens) return bad("page_tokens must be 16");
  if (c.max_seqs < 1 || c.max_seqs > kMaxSlots) return bad("max_seqs must be in 1..1024");
  if (c.max_seq_len < 2) return bad("bad max_seq_len");
  if (!attn_supported(c.dtype, c.head_dim, c.n_q_heads / c.n_kv_heads)) return bad("unsupported (head_dim, n_q/n_kv) combination");
  for (int i = 0; i < 2; ++i) if (c.reserved[i]) return bad("reserved fields must be 0");
  if (c.share_prompt_pages < 0 || c.share_prompt_pages > 2) return bad("share_prompt_pages must be 0, 1 or 2");
  if (c.share_prompt_pages == 2 && c.max_seq_len > 65535) return bad("share_prompt_pages = 2 needs max_seq_len <= 65535");
  if (c.attn_impl < 0 || c.attn_impl > 2) return bad("bad attn_impl");
  h->attn_impl = c.attn_impl == TANDEM_ATTN_AUTO ? (c.dtype == TANDEM_BF16 ? TANDEM_ATTN_MMA : TANDEM_ATTN_ALU) : c.attn_impl;
  if (h->attn_impl == TANDEM_ATTN_MMA && c.dtype != TANDEM_BF16) return bad("tensor-core attention needs bf16");
  if (cudaSetDevice(c.device) != cudaSuccess) { cudaGetLastError(); return bad("cudaSetDevice failed"); }
  h->esize = c.dtype == TANDEM_F32 ? 4 : 2;
  h->gemm_impl = c.gemm_impl == TANDEM_GEMM_AUTO ? (c.dtype == TANDEM_BF16 ? TANDEM_GEMM_TCGEN05 : TANDEM_GEMM_SIMT) : c.gemm_impl;
  if (h->gemm_impl == TANDEM_GEMM_TCGEN05 && c.dtype != TANDEM_BF16) return bad("tcgen05 GEMM needs bf16");
  h->row_cap = c.max_rows_per_step > 0 ? c.max_rows_per_step : 4096;
  h->row_cap = std::max(h->row_cap, c.max_seqs);   // every owned sequence must be able to decode in one step
  h->max_pages = (c.max_seq_len + kPageTokens - 1) / kPageTokens;
  h->tile_tok = std::max(1, kAttnTileRows / (c.n_q_heads / c.n_kv_heads));
  h->max_items = c.max_seqs * kAttnSplitTiles * (kAttnMaxSplits + 1) + h->row_cap;   // (q-tile, split) of short runs + the q-tiles of shared-prefix runs + q-tiles of longer ones
  h->max_comb = std::min(c.max_seqs * kAttnSplitTiles * h->tile_tok, h->row_cap);   // rows whose splits are combined
  h->part_cap = h->max_comb * (kAttnMaxSplits + 1);                 // (row, split) partials + one shared-prefix partial per row
  const int H = c.hidden, nq = c.n_q_heads, nkv = c.n_kv_heads, d = c.head_dim, I = c.intermediate, V = c.vocab, R = h->row_cap, S = c.max_seqs;
  const size_t page_bytes = (size_t)2 * c.n_layers * nkv * kPageTokens * d * h->esize;
  h->pool_pages = c.kv_bytes_per_model > 0 ? (int)std::min<int64_t>(c.kv_bytes_per_model / (int64_t)page_bytes, (int64_t)1 << 30)
                                           : S * h->max_pages + 1;
  if (h->pool_pages < 2) return bad("kv_bytes_per_model too small");
  h->slot_busy.assign(S, 0);

#define INIT_TRY(expr) do { int rc__ = (expr); if (rc__) { fprintf(stderr, "tandem_init: %s\n", h->err.c_str()); tandem_free(h); return rc__; } } while (0)
#define INIT_CU(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { fprintf(stderr, "tandem_init: %s: %s\n", #expr, cudaGetErrorString(e__)); tandem_free(h); return TANDEM_ECUDA; } } while (0)

  // sequence state
  INIT_TRY(dmalloc(h, &h->st_mem, (size_t)9 * S * 4));
  INIT_TRY(dmalloc(h, &h->st_mem8, (size_t)3 * S));
  INIT_CU(cudaMemset(h->st_mem, 0, (size_t)9 * S * 4));
  INIT_CU(cudaMemset(h->st_mem8, 0, (size_t)3 * S));
  {
    int32_t* p = h->st_mem;
    h->st.seq_id = p; p += S; h->st.prompt_len = p; p += S; h->st.n_ctx = p; p += S; h->st.ing[0] = p; p += S; h->st.ing[1] = p; p += S;
    h->st.cap_c = p; p += S; h->st.max_new = p; p += S; h->st.n_emit = p; p += S; h->st.grp = p; p += S;
    h->st.active = h->st_mem8; h->st.owner = h->st_mem8 + S; h->st.done = h->st_mem8 + 2 * S;
  }
  INIT_TRY(dmalloc(h, &h->tokens, (size_t)S * c.max_seq_len * 4));
  INIT_TRY(dmalloc(h, &h->out_owner, (size_t)S * c.max_seq_len));
  INIT_TRY(dmalloc(h, &h->out_logp, (size_t)S * c.max_seq_len * 4));
  INIT_CU(cudaMemset(h->tokens, 0, (size_t)S * c.max_seq_len * 4));
  INIT_TRY(dmalloc(h, &h->word_start_dev, (size_t)V));
  INIT_TRY(dmalloc(h, &h->stats, sizeof(DevStats)));
  INIT_CU(cudaMemset(h->stats, 0, sizeof(DevStats)));
  {
    int dev_sms = 0;
    if (cudaDeviceGetAttribute(&dev_sms, cudaDevAttrMultiProcessorCount, c.device) == cudaSuccess && dev_sms > 0) h->n_sms = dev_sms;
  }
  INIT_TRY(dmalloc(h, &h->work_ctr, (size_t)3 * c.n_layers * 4));   // [L] attention work counters, 2 x [L] for the profile mode's filtered launches
  INIT_CU(cudaMemset(h->work_ctr, 0, (size_t)3 * c.n_layers * 4));
  INIT_CU(cudaHostAlloc((void**)&h->oom_host, 4, cudaHostAllocMapped));
  *h->oom_host = 0;
  INIT_CU(cudaHostGetDevicePointer((void**)&h->oom_dev, h->oom_host, 0));
  INIT_CU(cudaHostAlloc((void**)&h->fault_host, 4, cudaHostAllocMapped));
  *h->fault_host = 0;
  INIT_CU(cudaHostGetDevicePointer((void**)&h->fault_dev, h->fault_host, 0));
  INIT_TRY(dmalloc(h, &h->n_active, 4));
  INIT_CU(cudaMemset(h->n_active, 0, 4));
  INIT_TRY(dmalloc(h, &h->stage_off, (size_t)(S + 1) * sizeof(long long)));
  INIT_TRY(dmalloc(h, &h->stage_i32, (size_t)5 * S * 4));

  // RoPE table: cos/sin of pos * theta^(-2j/d), evaluated in double, stored as fp32
  {
    const int half = d / 2;
    std::vector<float2> cs((size_t)c.max_seq_len * half);
    for (int j = 0; j < half; ++j) {
      const double inv = std::pow((double)c.rope_theta, -2.0 * j / d);
      for (int pos = 0; pos < c.max_seq_len; ++pos) {
        const double phi = (double)pos * inv;
        cs[(size_t)pos * half + j] = make_float2((float)std::cos(phi), (float)std::sin(phi));
      }
    }
    INIT_TRY(dmalloc(h, &h->rope_cs, cs.size() * sizeof(float2)));
    INIT_CU(cudaMemcpy(h->rope_cs, cs.data(), cs.size() * sizeof(float2), cudaMemcpyHostToDevice));
  }

  const int qkv_n = (nq + 2 * nkv) * d;
  // widest split-K partial buffer any GEMM needs, in floats per row (S*N); SIMT uses S = 1
  size_t cols = std::max({(size_t)qkv_n, (size_t)2 * I, (size_t)H});
  if (h->gemm_impl == TANDEM_GEMM_TCGEN05) {
    for (int nm = 1; nm <= 2; ++nm) {   // split counts are a function of the shape, the models per launch and the SM count
      cols = std::max(cols, (size_t)qkv_n * tc_gemm_splits(qkv_n, H, nm, h->n_sms));
      cols = std::max(cols, (size_t)H * tc_gemm_splits(H, nq * d, nm, h->n_sms));
      cols = std::max(cols, (size_t)H * tc_gemm_splits(H, I, nm, h->n_sms));
    }
  }
  h->gemm_out_cols = cols;
  if (h->gemm_impl == TANDEM_GEMM_TCGEN05 && h->esize == 2 && sk_applicable(2 * I, H, h->n_sms) && sk_gateup_init()) {
    // stream-K gate/up (gemm_streamk.cuh): one 256-row chunk of tail partials per CTA, flag / acknowledge counters (zero between launches)
    h->sk_rows = ((std::min(R, kTcMaxRows) + 31) / 32) * 32;
    INIT_TRY(dmalloc(h, &h->sk_scratch, (size_t)h->n_sms * 2 * h->sk_rows * kTcTileN * 4));
    INIT_TRY(dmalloc(h, &h->sk_flags, (size_t)2 * h->n_sms * 4));
    INIT_CU(cudaMemset(h->sk_flags, 0, (size_t)2 * h->n_sms * 4));
  }
  for (int m = 0; m < 2; ++m) {
    Workspace& w = h->ws[m];
    INIT_TRY(dmalloc(h, &w.x, (size_t)R * H * 4));
    INIT_TRY(dmalloc(h, &w.act, (size_t)R * H * h->esize));
    INIT_TRY(dmalloc(h, &w.q, (size_t)R * nq * d * 4));
    INIT_CU(cudaMemset(w.q, 0, (size_t)R * nq * d * 4));
    INIT_TRY(dmalloc(h, &w.attn_out, (size_t)R * nq * d * h->esize));
    INIT_TRY(dmalloc(h, &w.mlp_act, (size_t)R * I * h->esize));
    INIT_TRY(dmalloc(h, &w.lm_in, (size_t)std::max(S, 256) * H * h->esize));
    INIT_TRY(dmalloc(h, &w.gemm_out, (size_t)R * cols * 4));
    INIT_TRY(dmalloc(h, &w.logits, (size_t)S * V * 4));
    INIT_TRY(dmalloc(h, &w.chunk_part, (size_t)S * kSampleMaxChunks * 6 * 4));
    if (h->gemm_impl == TANDEM_GEMM_TCGEN05) INIT_TRY(dmalloc(h, &w.spart, (size_t)((V + kTcTileN - 1) / kTcTileN) * S * kTcSampleVals * 4));
    INIT_TRY(dmalloc(h, &w.chunk_ctr, (size_t)S * 4));
    INIT_CU(cudaMemset(w.chunk_ctr, 0, (size_t)S * 4));
    INIT_TRY(dmalloc(h, &w.part_acc, (size_t)h->part_cap * nq * d * 4));
    INIT_TRY(dmalloc(h, &w.part_ml, (size_t)h->part_cap * nq * sizeof(float2)));
    INIT_TRY(dmalloc(h, &w.kv, (size_t)h->pool_pages * page_bytes));
    // zero everything a TMA box or a padded MMA column may touch beyond the live rows
    INIT_CU(cudaMemset(w.act, 0, (size_t)R * H * h->esize));
    INIT_CU(cudaMemset(w.attn_out, 0, (size_t)R * nq * d * h->esize));
    INIT_CU(cudaMemset(w.mlp_act, 0, (size_t)R * I * h->esize));
    INIT_CU(cudaMemset(w.lm_in, 0, (size_t)std::max(S, 256) * H * h->esize));
    INIT_CU(cudaMemset(w.kv, 0, (size_t)h->pool_pages * page_bytes));
    // step tables
    const size_t tab_ints = (size_t)C_NUM + 5 * (size_t)R + (size_t)S + 5 * (size_t)h->max_items + 5 * (size_t)h->max_comb;
    INIT_TRY(dmalloc(h, &w.tab_mem, tab_ints * 4));
    INIT_CU(cudaMemset(w.tab_mem, 0, tab_ints * 4));
    {
      int32_t* p = w.tab_mem; StepTab& t = h->tab[m];
      t.counts = p; p += C_NUM; t.row_slot = p; p += R; t.row_pos = p; p += R; t.row_tok = p; p += R; t.row_kvslot = p; p += R; t.row_emit = p; p += R;
      t.emit_slot = p; p += S; t.item_row0 = p; p += h->max_items; t.item_ntok = p; p += h->max_items; t.item_kv0 = p; p += h->max_items;
      t.item_kv1 = p; p += h->max_items; t.item_part = p; p += h->max_items;
      t.comb_row = p; p += h->max_comb; t.comb_part0 = p; p += h->max_comb; t.comb_n = p; p += h->max_comb; t.comb_stride = p; p += h->max_comb; t.comb_gpart = p; p += h->max_comb;
    }
    // page tables
    INIT_TRY(dmalloc(h, &w.bt, (size_t)S * h->max_pages * 4));
    INIT_TRY(dmalloc(h, &w.npages, (size_t)2 * S * 4));   // npages, then nshared
    INIT_TRY(dmalloc(h, &w.free_pages, (size_t)h->pool_pages * 4));
    INIT_TRY(dmalloc(h, &w.free_top, 4));
    INIT_CU(cudaMemset(w.bt, 0, (size_t)S * h->max_pages * 4));
    h->pt[m].bt = w.bt; h->pt[m].npages = w.npages; h->pt[m].nshared = w.npages + S; h->pt[m].free_pages = w.free_pages; h->pt[m].free_top = w.free_top;
  }
  INIT_TRY(dmalloc(h, &h->gt_mem, (size_t)6 * S * 4));
  INIT_CU(cudaMemset(h->gt_mem, 0, (size_t)6 * S * 4));
  INIT_TRY(dmalloc(h, &h->gt_pages_mem, (size_t)2 * S * h->max_pages * 4));
  {
    int32_t* p = h->gt_mem;
    for (int m = 0; m < 2; ++m) { h->gt.state[m] = p; p += S; h->gt.donor[m] = p; p += S; h->gt.pages[m] = h->gt_pages_mem + (size_t)m * S * h->max_pages; }
    h->gt.npg = p; p += S; h->gt.ref = p; p += S;
  }
  INIT_CU(cudaEventCreateWithFlags(&h->ev_in, cudaEventDisableTiming));
  INIT_CU(cudaEventCreateWithFlags(&h->ev_out, cudaEventDisableTiming));
  INIT_CU(cudaStreamCreateWithFlags(&h->gs, cudaStreamNonBlocking));
  if (h->gemm_impl == TANDEM_GEMM_TCGEN05) {
    int cc_major = 0;
    cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, c.device);
    if (cc_major != 10) return bad("the tcgen05 GEMM needs an sm_100-class device (compute capability 10.x)");
  }
  if (h->gemm_impl == TANDEM_GEMM_TCGEN05 || h->attn_impl == TANDEM_ATTN_MMA) {
    h->tc = tc_gemm_create();
    if (!h->tc) { h->err = "tcgen05 GEMM setup failed (driver entry point for tensor maps not found)"; fprintf(stderr, "tandem_init: %s\n", h->err.c_str()); tandem_free(h); return TANDEM_ECUDA; }
  }
  if (cudaFuncSetAttribute(sample_switch_emit_kernel<256, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(NucleusSmem<256>)) != cudaSuccess)
    return bad("cannot reserve shared memory for the nucleus sampler");
  if (h->attn_impl == TANDEM_ATTN_MMA) {
    const long long total_rows = 2ll * c.n_layers * h->pool_pages * nkv * kPageTokens;
    if (total_rows >= (1ll << 31)) return bad("KV pool too large for the attention tensor map (2^31 rows)");
    for (int m = 0; m < 2; ++m) {
      const CUtensorMap* mp = tc_gemm_map(h->tc, h->ws[m].kv, (int)total_rows, d, kPageTokens);
      if (!mp) { h->err = "tensor map encode failed for the KV pool"; fprintf(stderr, "tandem_init: %s\n", h->err.c_str()); tandem_free(h); return TANDEM_ECUDA; }
      h->kv_map_store[m] = *mp;
      h->kv_map[m] = &h->kv_map_store[m];
    }
    {  // tcgen05 attention for scoring: q-tile boxes of 128 / G tokens x G heads x 64 dims; unsupported shapes keep the mma.sync kernel
      const int G = nq / nkv;
      Pair<AttnMmaArgs> dummy{}; Pair<CUtensorMap> dmaps{};
      bool ok = (d == 64 || d == 128) && G >= 1 && G <= 16 && run_attn_tc(dmaps, dmaps, dummy, d, G, 1, 0, true);
      for (int m = 0; m < 2 && ok; ++m) ok = tc_map_q3d(h->tc, &h->q_map_store[m], h->ws[m].q, d, nq, h->row_cap, G, kAtTileKv / G);
      if (!ok) cudaGetLastError();
      h->q_map_ok = ok;
    }
    Pair<AttnMmaArgs> dummy{}; Pair<CUtensorMap> dmaps{};
    if (!run_attn_mma(dmaps, dummy, d, nq / nkv, 1, 0, true)) {
      cudaGetLastError();
      h->err = "tensor-core attention: unsupported (head_dim, group) or shared-memory limit"; fprintf(stderr, "tandem_init: %s\n", h->err.c_str());
      tandem_free(h); return TANDEM_EINVAL;
    }
  }
  INIT_TRY(tandem_reset(h));
  *out = h;
  return TANDEM_OK;
}

int tandem_reset(tandem_handle* h) {
  if (!h) return TANDEM_EINVAL;
  const int S = h->cfg.max_seqs;
  CU(h, cudaDeviceSynchronize());
  CU(h, cudaMemset(h->st_mem8, 0, (size_t)3 * S));
  CU(h, cudaMemset(h->stats, 0, sizeof(DevStats)));
  CU(h, cudaMemset(h->n_active, 0, 4));
  if (h->oom_host) *h->oom_host = 0;
  std::vector<int32_t> fp(h->pool_pages);
  for (int i = 0; i < h->pool_pages - 1; ++i) fp[i] = h->pool_pages - 1 - i;   // pages 1..pool-1; popped in ascending order
  if (h->page_order_seed) {   // test hook: a seeded Fisher-Yates shuffle of the hand-out order (splitmix64)
    uint64_t x = h->page_order_seed;
    auto next = [&x]() { x += 0x9E3779B97F4A7C15ull; uint64_t z = x; z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; return z ^ (z >> 31); };
    for (int i = h->pool_pages - 2; i > 0; --i) std::swap(fp[i], fp[(size_t)(next() % (uint64_t)(i + 1))]);
  }
  const int32_t top = h->pool_pages - 1;
  for (int m = 0; m < 2; ++m) {
    CU(h, cudaMemcpy(h->ws[m].free_pages, fp.data(), (size_t)h->pool_pages * 4, cudaMemcpyHostToDevice));
    CU(h, cudaMemcpy(h->ws[m].free_top, &top, 4, cudaMemcpyHostToDevice));
    CU(h, cudaMemset(h->ws[m].npages, 0, (size_t)2 * S * 4));
    CU(h, cudaMemset(h->ws[m].chunk_ctr, 0, (size_t)S * 4));
  }
  std::fill(h->slot_busy.begin(), h->slot_busy.end(), 0);
  CU(h, cudaMemset(h->gt_mem, 0, (size_t)6 * S * 4));
  h->slot_grp.assign(S, -1); h->grp_live.assign(S, 0); h->grp_free.clear(); h->grp_reserved.assign(S, 0); h->grp_released = 0;
  for (int g = S - 1; g >= 0; --g) h->grp_free.push_back(g);
  h->launches = 0; h->preemptions = 0;
  return TANDEM_OK;
}

int tandem_get_stats(tandem_handle* h, tandem_stats* out) {
  if (!h || !out) return TANDEM_EINVAL;
  CU(h, cudaDeviceSynchronize());
  return fill_stats(h, out);
}

int tandem_set_profile(tandem_handle* h, int enable) {
  if (!h) return TANDEM_EINVAL;
  CU(h, cudaDeviceSynchronize());
  h->profile = enable != 0;
  if (enable) for (int i = 0; i < TANDEM_KC_NUM; ++i) { h->prof_ms[i] = 0.0; h->prof_n[i] = 0; }
  return TANDEM_OK;
}

int tandem_get_profile(tandem_handle* h, double* ms, int64_t* launches) {
  if (!h || !ms || !launches) return TANDEM_EINVAL;
  for (int i = 0; i < TANDEM_KC_NUM; ++i) { ms[i] = h->prof_ms[i]; launches[i] = h->prof_n[i]; }
  return TANDEM_OK;
}

const char* tandem_kernel_class_name(int kc) {
  static const char* names[TANDEM_KC_NUM] = {"sched", "embed_norm", "gemm_qkv", "rope_append", "attention", "attn_combine", "gemm_o",
                                             "residual_norm", "gemm_gateup", "swiglu", "gemm_down", "gemm_lmhead", "sample_switch_emit", "finalize", "score", "attention_catchup", "attention_empty"};
  return (kc >= 0 && kc < TANDEM_KC_NUM) ? names[kc] : "?";
}

int tandem_load_weights(tandem_handle* h, int model, const tandem_weights* w) {
  if (!h || !w || model < 0 || model > 1) return fail(h, TANDEM_EINVAL, "bad arguments");
  const tandem_config& c = h->cfg;
  const size_t es = h->esize;
  const int H = c.hidden, nq = c.n_q_heads, nkv = c.n_kv_heads, d = c.head_dim, I = c.intermediate, V = c.vocab, L = c.n_layers;
  if (!w->embed || !w->lm_head || !w->final_norm || !w->attn_norm || !w->wq || !w->wk || !w->wv || !w->wo || !w->mlp_norm || !w->w_gate || !w->w_up || !w->w_down)
    return fail(h, TANDEM_EINVAL, "NULL weight pointer");
  ModelWeights& mw = h->w[model];
  const cudaMemcpyKind kind = w->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  auto put = [&](void** dst, size_t dst_off_elems, const void* src, size_t elems, size_t total_elems) -> int {
    if (!src) return fail(h, TANDEM_EINVAL, "NULL layer weight pointer");
    if (!*dst) DM(h, (char**)dst, total_elems * es);
    CU(h, cudaMemcpy((char*)*dst + dst_off_elems * es, src, elems * es, kind));
    return TANDEM_OK;
  };
  int rc;
  CU(h, cudaDeviceSynchronize());
  if ((rc = put(&mw.embed, 0, w->embed, (size_t)V * H, (size_t)V * H))) return rc;
  if ((rc = put(&mw.lm_head, 0, w->lm_head, (size_t)V * H, (size_t)V * H))) return rc;
  if ((rc = put(&mw.final_norm, 0, w->final_norm, H, H))) return rc;
  mw.attn_norm.resize(L, nullptr); mw.wqkv.resize(L, nullptr); mw.wo.resize(L, nullptr); mw.mlp_norm.resize(L, nullptr); mw.wgu.resize(L, nullptr); mw.wdown.resize(L, nullptr);
  const size_t qn = (size_t)nq * d * H, kn = (size_t)nkv * d * H;
  for (int l = 0; l < L; ++l) {
    if ((rc = put(&mw.attn_norm[l], 0, w->attn_norm[l], H, H))) return rc;
    if ((rc = put(&mw.wqkv[l], 0, w->wq[l], qn, qn + 2 * kn))) return rc;            // [q | k | v] rows
    if ((rc = put(&mw.wqkv[l], qn, w->wk[l], kn, qn + 2 * kn))) return rc;
    if ((rc = put(&mw.wqkv[l], qn + kn, w->wv[l], kn, qn + 2 * kn))) return rc;
    if ((rc = put(&mw.wo[l], 0, w->wo[l], (size_t)H * nq * d, (size_t)H * nq * d))) return rc;
    if ((rc = put(&mw.mlp_norm[l], 0, w->mlp_norm[l], H, H))) return rc;
    if (h->gemm_impl == TANDEM_GEMM_TCGEN05) {   // rows interleaved: 2i = gate_i, 2i+1 = up_i (SwiGLU runs in the GEMM epilogue)
      if (!w->w_gate[l] || !w->w_up[l]) return fail(h, TANDEM_EINVAL, "NULL layer weight pointer");
      if (!mw.wgu[l]) DM(h, (char**)&mw.wgu[l], (size_t)2 * I * H * es);
      CU(h, cudaMemcpy2D(mw.wgu[l], (size_t)2 * H * es, w->w_gate[l], (size_t)H * es, (size_t)H * es, I, kind));
      CU(h, cudaMemcpy2D((char*)mw.wgu[l] + (size_t)H * es, (size_t)2 * H * es, w->w_up[l], (size_t)H * es, (size_t)H * es, I, kind));
    } else {
      if ((rc = put(&mw.wgu[l], 0, w->w_gate[l], (size_t)I * H, (size_t)2 * I * H))) return rc;   // [gate | up] rows
      if ((rc = put(&mw.wgu[l], (size_t)I * H, w->w_up[l], (size_t)I * H, (size_t)2 * I * H))) return rc;
    }
    if ((rc = put(&mw.wdown[l], 0, w->w_down[l], (size_t)H * I, (size_t)H * I))) return rc;
  }
  CU(h, cudaDeviceSynchronize());
  mw.loaded = true;
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; h->gkey.valid = false; }
  if (h->tc) tc_gemm_invalidate(h->tc, model);
  return TANDEM_OK;
}

int tandem_step(tandem_handle* h, const tandem_step_in* in, tandem_step_out* out, void* cuda_stream) {
  int rc = check_ready(h);
  if (rc) return rc;
  if (!in) return fail(h, TANDEM_EINVAL, "step_in is NULL");
  if ((rc = check_params(h, in->params))) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if ((rc = check_oom_flag(h))) return rc;
  if ((rc = sync_word_start(h, in->params, s))) return rc;
  if (in->n_admit > 0) {
    if ((rc = check_oom(h, s))) return rc;
    if ((rc = refresh_slots(h, s))) return rc;
    if ((rc = admit(h, in->params, in->ovr, in->n_admit, in->admit_tokens, in->admit_offsets, in->admit_seq_id, in->admit_max_new,
                    out ? out->admit_slots : nullptr, s))) return rc;
  }
  return run_step(h, make_io(out, in->ovr), make_rule(in->params), s);
}

int tandem_evict(tandem_handle* h, int32_t slot, void* cuda_stream) {
  if (!h) return TANDEM_EINVAL;
  if (h->cuda_fault) return fail(h, TANDEM_ECUDA, "a previous CUDA error is sticky: " + h->err);
  if (slot < 0 || slot >= h->cfg.max_seqs) return fail(h, TANDEM_EINVAL, "slot out of range");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int rc = refresh_slots(h, s);
  if (rc) return rc;
  if (!h->slot_busy[slot]) return fail(h, TANDEM_EINVAL, "slot holds no sequence");
  if ((rc = preempt_slot(h, slot, s))) return rc;
  if (h->oom_host) *h->oom_host = 0;             // pages came back: a stall or dead lock reported so far is history
  CU(h, cudaMemset(&h->stats->err_oom, 0, sizeof(int)));
  return TANDEM_OK;
}

int tandem_generate(tandem_handle* h, const tandem_params* params, int32_t B, const int32_t* prompt_tokens, const int64_t* prompt_offsets,
                    const int32_t* max_new, const int32_t* seq_ids, const tandem_overrides* ovr, int32_t out_stride, int32_t* out_tokens,
                    uint8_t* out_owner, float* out_sen_logp, int32_t* out_len, tandem_stats* stats, void* cuda_stream) {
  int rc = check_ready(h);
  if (rc) return rc;
  if ((rc = check_params(h, params))) return rc;
  if (B < 0 || (B > 0 && (!prompt_tokens || !prompt_offsets || !max_new || !out_len))) return fail(h, TANDEM_EINVAL, "bad arguments");
  const tandem_config& c = h->cfg;
  if (ovr && B > c.max_seqs) return fail(h, TANDEM_EINVAL, "overrides need B <= max_seqs (rows are addressed by slot)");
  for (int b = 0; b < B; ++b) if (max_new[b] > out_stride) return fail(h, TANDEM_EINVAL, "out_stride < max_new");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if ((rc = tandem_reset(h))) return rc;
  if ((rc = sync_word_start(h, params, s))) return rc;
  if (out_tokens) std::memset(out_tokens, 0, (size_t)B * out_stride * 4);
  if (out_owner) std::memset(out_owner, 0, (size_t)B * out_stride);
  if (out_sen_logp) std::memset(out_sen_logp, 0, (size_t)B * out_stride * 4);
  EventPair ev;
  CU(h, cudaEventCreate(&ev.e0)); CU(h, cudaEventCreate(&ev.e1));
  CU(h, cudaEventRecord(ev.e0, s));
  const StepIO io = make_io(nullptr, ovr);
  const RuleParams rp = make_rule(params);
  // Continuous batching: a sequence is admitted on its CURRENT need - the pages of
  // its prompt in both pools - plus a watermark (the pages every resident sequence can grow by until the next poll), not on
  // prompt + max_new. Pages come from the device-side free stacks on demand; when a pool runs dry the scheduler stalls the
  // sequences it cannot serve (nothing is corrupted) and the host preempts the youngest resident sequence: its pages are freed,
  // it goes back to the head of the queue and is redone from its prompt - bit-identically, since every random draw is addressed
  // by (seed, seq_id, t, vocabulary id) and no result depends on the batch composition.
  std::vector<int> slot_seq(c.max_seqs, -1);
  std::vector<int32_t> nemit(c.max_seqs), plen(c.max_seqs);
  auto prompt_pages = [&](int b) { return (int)((prompt_offsets[b + 1] - prompt_offsets[b] + kPageTokens - 1) / kPageTokens) + 1; };
  auto total_pages = [&](int b) { return (int)((prompt_offsets[b + 1] - prompt_offsets[b] + max_new[b] + kPageTokens - 1) / kPageTokens); };
  auto shared_pages_of = [&](int b) { return (int)((prompt_offsets[b + 1] - prompt_offsets[b] - 1) / kPageTokens); };
  auto same_prompt = [&](int a, int b) {
    const int64_t la = prompt_offsets[a + 1] - prompt_offsets[a], lb = prompt_offsets[b + 1] - prompt_offsets[b];
    return la == lb && std::memcmp(prompt_tokens + prompt_offsets[a], prompt_tokens + prompt_offsets[b], (size_t)la * 4) == 0;
  };
  const int pages_avail = h->pool_pages - 1;
  for (int b = 0; b < B; ++b) if (total_pages(b) > pages_avail) return fail(h, TANDEM_ENOMEM, "a single sequence needs more KV pages than the pool holds");
  std::vector<int> requeue;               // preempted sequences, admitted before the rest of the queue
  int next = 0, finished = 0, resident = 0;
  const int max_poll = 16;
  int64_t budget = 0;   // generous bound on the number of steps: guards against a stuck sequence
  for (int b = 0; b < B; ++b) budget += max_new[b] + (prompt_offsets[b + 1] - prompt_offsets[b]) / std::max(1, h->row_cap / 4) + 4;
  budget = 8 * budget + 4096;
  int free_pages_now = pages_avail;       // min over the two pools, as of the last poll
  bool starving = false;
  while (finished < B) {
    // ---- admission
    const int growth = max_poll / kPageTokens + 1;                // pages a resident sequence may take per model until the next poll
    int nfree = 0;
    for (int i = 0; i < c.max_seqs; ++i) nfree += !h->slot_busy[i];
    // what the resident sequences may still take until the next poll (never more than the rest of their context)
    int avail = free_pages_now;
    for (int i = 0; i < c.max_seqs; ++i)
      if (slot_seq[i] >= 0) {
        const int b = slot_seq[i];
        const int held = (int)((prompt_offsets[b + 1] - prompt_offsets[b] + nemit[i] + kPageTokens - 1) / kPageTokens);
        avail -= std::min(growth, std::max(0, total_pages(b) - held));
      }
    auto admit_need = [&](int b) { return std::min(prompt_pages(b) + growth, total_pages(b)); };
    if (!starving) {
      while (!requeue.empty() && nfree > 0 && (avail >= admit_need(requeue.back()) || resident == 0)) {
        const int b = requeue.back(); requeue.pop_back();
        int32_t slot = -1; const int32_t id = seq_ids ? seq_ids[b] : b;
        if ((rc = admit(h, params, ovr, 1, prompt_tokens, prompt_offsets + b, &id, max_new + b, &slot, s))) return rc;
        slot_seq[slot] = b; --nfree; ++resident; avail -= admit_need(b);
      }
      int n = 0;
      while (requeue.empty() && n < std::min(nfree, B - next)) {
        const int b = next + n;
        const int need = admit_need(b) - ((c.share_prompt_pages && n > 0 && same_prompt(b - 1, b)) ? std::min(shared_pages_of(b), admit_need(b)) : 0);
        if (avail < need && resident + n > 0) break;              // an empty engine always takes the next sequence (it fits: checked above)
        avail -= need; ++n;
      }
      if (ovr && next == 0 && n < B) return fail(h, TANDEM_ENOMEM, "overrides are addressed by slot = batch index: the whole batch must fit the KV pools at once");
      if (n > 0) {
        std::vector<int32_t> slots(n), ids(n);
        for (int i = 0; i < n; ++i) ids[i] = seq_ids ? seq_ids[next + i] : next + i;
        if ((rc = admit(h, params, ovr, n, prompt_tokens, prompt_offsets + next, ids.data(), max_new + next, slots.data(), s))) return rc;
        for (int i = 0; i < n; ++i) slot_seq[slots[i]] = next + i;
        next += n; resident += n;
      }
    }
    // ---- steps until the next poll: no longer than the soonest possible finish when there is no EOS to end a sequence early
    int poll = starving ? 2 : max_poll;
    if (params->eos_id < 0) {
      int soonest = max_poll;
      for (int i = 0; i < c.max_seqs; ++i) if (slot_seq[i] >= 0) soonest = std::min(soonest, std::max(1, max_new[slot_seq[i]] - nemit[i]));
      poll = std::min(poll, soonest);
    }
    if ((budget -= poll) < 0) return fail(h, TANDEM_ESTATE, "generation made no progress (internal error)");
    for (int k = 0; k < poll; ++k) if ((rc = run_step(h, io, rp, s))) return rc;
    if ((rc = refresh_slots(h, s))) return rc;                   // synchronises the stream
    CU(h, cudaMemcpy(nemit.data(), h->st.n_emit, (size_t)c.max_seqs * 4, cudaMemcpyDeviceToHost));
    CU(h, cudaMemcpy(plen.data(), h->st.prompt_len, (size_t)c.max_seqs * 4, cudaMemcpyDeviceToHost));
    {
      int32_t ft[2];
      for (int m = 0; m < 2; ++m) CU(h, cudaMemcpy(&ft[m], h->ws[m].free_top, 4, cudaMemcpyDeviceToHost));
      free_pages_now = std::min(ft[0], ft[1]);
    }
    // ---- finished sequences: results to the caller's buffers
    for (int i = 0; i < c.max_seqs; ++i) {
      if (slot_seq[i] < 0 || h->slot_busy[i]) continue;
      const int b = slot_seq[i], len = nemit[i];
      out_len[b] = len;
      if (out_tokens) CU(h, cudaMemcpy(out_tokens + (size_t)b * out_stride, h->tokens + (size_t)i * c.max_seq_len + plen[i], (size_t)len * 4, cudaMemcpyDeviceToHost));
      if (out_owner) CU(h, cudaMemcpy(out_owner + (size_t)b * out_stride, h->out_owner + (size_t)i * c.max_seq_len, (size_t)len, cudaMemcpyDeviceToHost));
      if (out_sen_logp) CU(h, cudaMemcpy(out_sen_logp + (size_t)b * out_stride, h->out_logp + (size_t)i * c.max_seq_len, (size_t)len * 4, cudaMemcpyDeviceToHost));
      slot_seq[i] = -1; nemit[i] = 0;
      ++finished; --resident;
    }
    // ---- a pool ran dry since the last poll: preempt the youngest resident sequence (the least work to redo)
    starving = false;
    if (h->oom_host && *(volatile int32_t*)h->oom_host) {
      *h->oom_host = 0;
      CU(h, cudaMemset(&h->stats->err_oom, 0, sizeof(int)));
      if (resident > 0) {
        if (ovr) return fail(h, TANDEM_ENOMEM, "KV pool exhausted and overrides are addressed by slot: a sequence cannot be preempted");
        int victim = -1;
        for (int i = 0; i < c.max_seqs; ++i)
          if (slot_seq[i] >= 0 && (victim < 0 || nemit[i] < nemit[victim] || (nemit[i] == nemit[victim] && slot_seq[i] > slot_seq[victim]))) victim = i;
        if (resident == 1) return fail(h, TANDEM_ENOMEM, "KV pool exhausted by a single sequence (internal error: its whole context was checked to fit)");
        if ((rc = preempt_slot(h, victim, s))) return rc;
        requeue.push_back(slot_seq[victim]);
        slot_seq[victim] = -1; nemit[victim] = 0; --resident;
        ++h->preemptions;
        starving = true;                    // poll soon: more may have to go before the stalled sequences move again
        for (int m = 0; m < 2; ++m) { int32_t ft; CU(h, cudaMemcpy(&ft, h->ws[m].free_top, 4, cudaMemcpyDeviceToHost)); free_pages_now = m ? std::min(free_pages_now, ft) : ft; }
      }
    }
  }
  CU(h, cudaEventRecord(ev.e1, s));
  CU(h, cudaEventSynchronize(ev.e1));
  float ms = 0.f;
  CU(h, cudaEventElapsedTime(&ms, ev.e0, ev.e1));
  if ((rc = check_oom(h, s))) return rc;
  if (stats) {
    if ((rc = fill_stats(h, stats))) return rc;
    stats->seconds_total = ms * 1e-3;
  }
  return TANDEM_OK;
}

int tandem_score(tandem_handle* h, int32_t n_seqs, const int32_t* tokens, const int64_t* offsets, float temperature,
                 float* sen_logp, float* jun_logp, float* overlap, tandem_stats* stats, void* cuda_stream) {
  int rc = check_ready(h);
  if (rc) return rc;
  if (n_seqs < 0 || (n_seqs > 0 && (!tokens || !offsets))) return fail(h, TANDEM_EINVAL, "bad arguments");
  if (!(temperature > 0.f)) return fail(h, TANDEM_EINVAL, "temperature must be > 0");
  const tandem_config& c = h->cfg;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  for (int m = 0; m < 2; ++m) {   // the scoring buffers exist from the first call on
    if (!h->ws[m].score_lm_in) DM(h, &h->ws[m].score_lm_in, (size_t)h->row_cap * c.hidden * h->esize);
    if (!h->ws[m].score_logits) DM(h, &h->ws[m].score_logits, (size_t)h->row_cap * c.vocab * sizeof(float));
    if (!h->score_out[m]) DM(h, &h->score_out[m], (size_t)c.max_seqs * c.max_seq_len * sizeof(float));
  }
  if ((rc = tandem_reset(h))) return rc;
  const int64_t total = n_seqs > 0 ? offsets[n_seqs] - offsets[0] : 0;
  for (float* o : {sen_logp, jun_logp, overlap}) if (o && total > 0) std::memset(o + offsets[0], 0, (size_t)total * sizeof(float));
  EventPair ev;
  CU(h, cudaEventCreate(&ev.e0)); CU(h, cudaEventCreate(&ev.e1));
  CU(h, cudaEventRecord(ev.e0, s));
  tandem_params prm{};   // admission only needs an owner; the rule never runs while scoring
  prm.p = 0.f; prm.switch_mode = TANDEM_TOGGLE; prm.start_owner = TANDEM_SENIOR; prm.temperature = temperature; prm.top_p = 1.f; prm.top_k = 0; prm.eos_id = -1;
  const StepIO io = make_io(nullptr, nullptr);
  const RuleParams rp = make_rule(&prm);
  auto pages_of = [&](int b) { return (int)((offsets[b + 1] - offsets[b] + kPageTokens - 1) / kPageTokens); };
  const int pages_avail = h->pool_pages - 1;
  for (int b = 0; b < n_seqs; ++b) {
    if (offsets[b + 1] - offsets[b] < 1) return fail(h, TANDEM_EINVAL, "empty stream");
    if (pages_of(b) > pages_avail) return fail(h, TANDEM_ENOMEM, "a single stream needs more KV pages than the pool holds");
  }
  std::vector<int> slot_seq(c.max_seqs, -1), slot_pages(c.max_seqs, 0);
  std::vector<int32_t> ids(c.max_seqs), ones(c.max_seqs, 1);
  std::vector<float> row(c.max_seq_len);
  int next = 0, finished = 0, pages_reserved = 0;
  int64_t budget = 1024;
  for (int b = 0; b < n_seqs; ++b) budget += 4 + 4 * (offsets[b + 1] - offsets[b]);
  while (finished < n_seqs) {
    if (--budget < 0) return fail(h, TANDEM_ESTATE, "scoring made no progress (internal error)");
    int nfree = 0;
    for (int i = 0; i < c.max_seqs; ++i) nfree += !h->slot_busy[i];
    int n = 0, add = 0;
    while (n < std::min(nfree, n_seqs - next) && pages_reserved + add + pages_of(next + n) <= pages_avail) { add += pages_of(next + n); ++n; }
    if (n > 0) {
      std::vector<int32_t> slots(n);
      for (int i = 0; i < n; ++i) ids[i] = next + i;
      if ((rc = admit(h, &prm, nullptr, n, tokens, offsets + next, ids.data(), ones.data(), slots.data(), s, true))) return rc;
      for (int i = 0; i < n; ++i) { slot_seq[slots[i]] = next + i; slot_pages[slots[i]] = pages_of(next + i); }
      pages_reserved += add;
      next += n;
    }
    if (h->profile) { h->ev_used = 0; h->prof_pending.clear(); }
    h->scoring = true;
    rc = launch_step(h, io, rp, s, true, 1.f / temperature);
    h->scoring = false;
    if (rc) return rc;
    CU(h, cudaGetLastError());
    if ((rc = refresh_slots(h, s))) return rc;   // synchronises the stream
    if (h->profile) {
      for (const auto& r : h->prof_pending) {
        float pms = 0.f;
        CU(h, cudaEventElapsedTime(&pms, r.e0, r.e1));
        h->prof_ms[r.cls] += pms; h->prof_n[r.cls] += 1;
      }
    }
    for (int i = 0; i < c.max_seqs; ++i) {
      if (slot_seq[i] < 0 || h->slot_busy[i]) continue;
      const int b = slot_seq[i];
      const int64_t len = offsets[b + 1] - offsets[b];
      float* outs[3] = {sen_logp, jun_logp, overlap};
      const float* devs[3] = {h->out_logp, h->score_out[0], h->score_out[1]};
      for (int k = 0; k < 3; ++k) {
        if (!outs[k] || len < 2) continue;
        CU(h, cudaMemcpy(outs[k] + offsets[b] + 1, devs[k] + (size_t)i * c.max_seq_len + 1, (size_t)(len - 1) * sizeof(float), cudaMemcpyDeviceToHost));
      }
      slot_seq[i] = -1;
      pages_reserved -= slot_pages[i]; slot_pages[i] = 0;
      ++finished;
    }
  }
  CU(h, cudaEventRecord(ev.e1, s));
  CU(h, cudaEventSynchronize(ev.e1));
  float ms = 0.f;
  CU(h, cudaEventElapsedTime(&ms, ev.e0, ev.e1));
  if ((rc = check_oom(h, s))) return rc;
  if (stats) {
    if ((rc = fill_stats(h, stats))) return rc;
    stats->seconds_total = ms * 1e-3;
  }
  return TANDEM_OK;
}

int tandem_grpo_objective(int32_t n_groups, int32_t group, int32_t stride, const float* rewards, const int32_t* len, const uint8_t* owner,
                          const float* logp_new, const float* logp_old, const float* logp_ref, float clip_eps, float kl_beta, float adv_eps,
                          float* advantages, float* token_obj, float* seq_obj, float* result, void* cuda_stream) {
  if (n_groups < 0 || group < 1 || stride < 1 || !(clip_eps >= 0.f) || !(adv_eps >= 0.f)) return TANDEM_EINVAL;
  if (!rewards || !len || !owner || !logp_new || !logp_old || !advantages || !seq_obj || !result) return TANDEM_EINVAL;
  if (kl_beta != 0.f && !logp_ref) return TANDEM_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int B = n_groups * group;
  if (cudaMemsetAsync(result, 0, 8 * sizeof(float), s) != cudaSuccess) { cudaGetLastError(); return TANDEM_ECUDA; }
  if (B == 0) return TANDEM_OK;
  const GrpoArgs a{B, group, stride, rewards, len, owner, logp_new, logp_old, logp_ref, clip_eps, kl_beta, adv_eps, advantages, token_obj, seq_obj, result};
  grpo_seq_kernel<256><<<B, 256, 0, s>>>(a);
  return cudaGetLastError() == cudaSuccess ? TANDEM_OK : TANDEM_ECUDA;
}

// ---------------------------------------------------------------------------------------------- tandem_grpo_objective_static
// The GRPO objective for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
// grpo_seq_kernel's scratch - the arrival counters, the per-rollout objectives the last CTA reduces in index order, the advantages -
// lives in ONE file-scope device array instead of caller-provided buffers. Every GPU that loads the library holds its kGrpoStaticBytes
// (65,792 bytes) until the process exits. Layout (floats): [0, 8) result + counters (zeroed by every call), [64, 64 + MAX) per-rollout
// objectives, [64 + MAX, 64 + 2 MAX) advantages; entries [0, B) of both are written before the last CTA reads them, the rest keeps the
// previous call's values and is never read. All calls share the array: two calls that overlap on the GPU (different streams, or
// different host threads without ordering) race on it.
constexpr int kGrpoStaticMaxSeqs = TANDEM_GRPO_STATIC_MAX_ROLLOUTS;
constexpr int kGrpoStaticHead = 64;                                           // floats in front of the per-rollout arrays
constexpr size_t kGrpoStaticBytes = (size_t)(kGrpoStaticHead + 2 * kGrpoStaticMaxSeqs) * sizeof(float);
static __device__ __align__(256) unsigned char g_grpo_static_scratch[kGrpoStaticBytes];

namespace {
// In host code `g_grpo_static_scratch` is a host-side stand-in, not a device address: the kernel gets the address
// cudaGetSymbolAddress returns for the CURRENT device, looked up once per device.
constexpr int kMaxDevices = 64;
std::mutex g_grpo_static_mu;
float* g_grpo_static_ptr[kMaxDevices] = {};
int grpo_static_scratch(float** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return TANDEM_ECUDA; }
  std::lock_guard<std::mutex> lk(g_grpo_static_mu);
  if (!g_grpo_static_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_grpo_static_scratch);
    if (e != cudaSuccess || !p) {
      fprintf(stderr, "tandem_grpo_objective_static: cudaGetSymbolAddress failed on device %d: %s\n", dev, cudaGetErrorString(e));
      cudaGetLastError();
      return TANDEM_ECUDA;
    }
    g_grpo_static_ptr[dev] = (float*)p;
  }
  *out = g_grpo_static_ptr[dev];
  return TANDEM_OK;
}
}  // namespace

int tandem_grpo_objective_static(int32_t n_groups, int32_t group, int32_t stride, const float* rewards, const int32_t* len, const uint8_t* owner,
                                 const float* logp_new, const float* logp_old, const float* logp_ref, float clip_eps, float kl_beta, float adv_eps,
                                 float* token_obj, float* result4, void* cuda_stream) {
  if (n_groups < 0 || group < 1 || stride < 1 || !(clip_eps >= 0.f) || !(adv_eps >= 0.f)) return TANDEM_EINVAL;
  if (!rewards || !len || !owner || !logp_new || !logp_old || !result4) return TANDEM_EINVAL;
  if (kl_beta != 0.f && !logp_ref) return TANDEM_EINVAL;
  const long long B = (long long)n_groups * group;
  if (B > kGrpoStaticMaxSeqs) {
    fprintf(stderr, "tandem_grpo_objective_static: %lld rollouts exceed the static scratch (TANDEM_GRPO_STATIC_MAX_ROLLOUTS = %d); use tandem_grpo_objective\n",
            B, kGrpoStaticMaxSeqs);
    return TANDEM_EINVAL;
  }
  float* scratch = nullptr;
  const int rc = grpo_static_scratch(&scratch);
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (cudaMemsetAsync(scratch, 0, 8 * sizeof(float), s) != cudaSuccess) { cudaGetLastError(); return TANDEM_ECUDA; }   // results and counters start at zero
  if (B > 0) {
    const GrpoArgs a{(int)B, group, stride, rewards, len, owner, logp_new, logp_old, logp_ref, clip_eps, kl_beta, adv_eps,
                     scratch + kGrpoStaticHead + kGrpoStaticMaxSeqs, token_obj, scratch + kGrpoStaticHead, scratch};
    grpo_seq_kernel<256><<<(int)B, 256, 0, s>>>(a);
    if (cudaGetLastError() != cudaSuccess) return TANDEM_ECUDA;
  }
  if (cudaMemcpyAsync(result4, scratch, 4 * sizeof(float), cudaMemcpyDeviceToDevice, s) != cudaSuccess) { cudaGetLastError(); return TANDEM_ECUDA; }
  return TANDEM_OK;
}

void tandem_free(tandem_handle* h) {
  if (!h) return;
  cudaDeviceSynchronize();
  if (h->graph) cudaGraphExecDestroy(h->graph);
  if (h->tc) tc_gemm_destroy(h->tc);
  auto fr = [](void* p) { if (p) cudaFree(p); };
  for (int m = 0; m < 2; ++m) {
    Workspace& w = h->ws[m];
    fr(w.score_lm_in); fr(w.score_logits); fr(w.spart); fr(w.chunk_part); fr(w.chunk_ctr); fr(w.x); fr(w.act); fr(w.q); fr(w.attn_out); fr(w.mlp_act); fr(w.lm_in); fr(w.gemm_out); fr(w.logits); fr(w.part_acc); fr(w.part_ml); fr(w.kv);
    fr(w.tab_mem); fr(w.bt); fr(w.npages); fr(w.free_pages); fr(w.free_top);
    ModelWeights& mw = h->w[m];
    fr(mw.embed); fr(mw.lm_head); fr(mw.final_norm);
    for (auto* v : {&mw.attn_norm, &mw.wqkv, &mw.wo, &mw.mlp_norm, &mw.wgu, &mw.wdown}) for (void* p : *v) fr(p);
  }
  for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
  if (h->ev_in) cudaEventDestroy(h->ev_in);
  if (h->ev_out) cudaEventDestroy(h->ev_out);
  if (h->gs) cudaStreamDestroy(h->gs);
  fr(h->score_out[0]); fr(h->score_out[1]); fr(h->st_mem); fr(h->st_mem8); fr(h->tokens); fr(h->out_owner); fr(h->out_logp); fr(h->rope_cs); fr(h->word_start_dev); fr(h->stats);
  fr(h->gt_mem); fr(h->gt_pages_mem);
  if (h->oom_host) cudaFreeHost(h->oom_host);
  if (h->fault_host) cudaFreeHost(h->fault_host);
  if (h->sk_scratch) cudaFree(h->sk_scratch);
  if (h->sk_flags) cudaFree(h->sk_flags);
  fr(h->n_active); fr(h->work_ctr); fr(h->stage_tokens); fr(h->stage_off); fr(h->stage_i32);
  cudaGetLastError();
  delete h;
}

const char* tandem_last_error(const tandem_handle* h) { return h ? h->err.c_str() : "NULL handle"; }

// ---------------------------------------------------------------------------------------------- test hooks
__global__ void test_uniforms_kernel(unsigned long long seed, int seq_id, int t, int stream, int n, float* out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (stream == 1) { out[i] = u_switch_counter(seed, seq_id, i); return; }
  uint32_t c[4] = {(uint32_t)(i >> 2), (uint32_t)t, (uint32_t)seq_id, 0u};
  philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
  out[i] = uniform_from_bits(c[i & 3]);
}
__global__ void test_philox_kernel(uint32_t* io) {
  uint32_t c[4] = {io[0], io[1], io[2], io[3]};
  philox4x32_10(c, io[4], io[5]);
  for (int i = 0; i < 4; ++i) io[6 + i] = c[i];
}

int tandem_test_uniforms(uint64_t seed, int32_t seq_id, int32_t t, int32_t stream, int32_t n, float* out_dev) {
  if (n <= 0 || !out_dev) return TANDEM_EINVAL;
  test_uniforms_kernel<<<(n + 255) / 256, 256>>>(seed, seq_id, t, stream, n, out_dev);
  return cudaDeviceSynchronize() == cudaSuccess ? TANDEM_OK : TANDEM_ECUDA;
}

int tandem_test_nucleus(int32_t vocab, float temperature, float top_p, int32_t top_k, const float* logits_dev, const float* u_dev, int32_t* token_dev,
                        uint8_t* keep_dev) {
  if (vocab <= 0 || !(temperature > 0.f) || !(top_p > 0.f && top_p <= 1.f) || top_k > kNucleusCap || !logits_dev || !u_dev || !token_dev || !keep_dev) return TANDEM_EINVAL;
  cudaFuncSetAttribute(test_nucleus_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(NucleusSmem<256>));
  test_nucleus_kernel<256><<<1, 256, sizeof(NucleusSmem<256>)>>>(logits_dev, vocab, temperature, top_p, top_k, u_dev, token_dev, keep_dev);
  return cudaDeviceSynchronize() == cudaSuccess ? TANDEM_OK : TANDEM_ECUDA;
}

int tandem_test_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t* d = nullptr;
  if (cudaMalloc(&d, 40) != cudaSuccess) return TANDEM_ENOMEM;
  uint32_t hbuf[10] = {ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1], 0, 0, 0, 0};
  cudaMemcpy(d, hbuf, 40, cudaMemcpyHostToDevice);
  test_philox_kernel<<<1, 1>>>(d);
  const cudaError_t e = cudaMemcpy(hbuf, d, 40, cudaMemcpyDeviceToHost);
  cudaFree(d);
  for (int i = 0; i < 4; ++i) out[i] = hbuf[6 + i];
  return e == cudaSuccess ? TANDEM_OK : TANDEM_ECUDA;
}

int tandem_test_gemm(int32_t dtype, int32_t impl, int32_t rows, int32_t N, int32_t K, const void* A_dev, const void* W_dev, float* out_dev) {
  if (rows < 0 || N <= 0 || K <= 0 || !A_dev || !W_dev || !out_dev) return TANDEM_EINVAL;
  if (impl == TANDEM_GEMM_TCGEN05 || (impl >= 3 && impl <= 5)) {   // 3: SwiGLU epilogue; 4, 5: the same two as CTA pairs (cta_group::2)
    if (dtype != TANDEM_BF16) return TANDEM_EINVAL;
    return tc_gemm_test(rows, N, K, A_dev, W_dev, out_dev, (impl == 3 || impl == 5) ? kTcEpiSwiGLU : kTcEpiPartial, impl >= 4);
  }
  dim3 grid((N + kSimtTile - 1) / kSimtTile, std::max(1, std::min((rows + kSimtTile - 1) / kSimtTile, 64)));
  if (dtype == TANDEM_F32) {
    Pair<SimtGemmArgs<float>> g; g.m[0] = g.m[1] = SimtGemmArgs<float>{nullptr, rows, (const float*)A_dev, (const float*)W_dev, out_dev, N, K};
    gemm_simt_kernel<float><<<grid, 256>>>(g);
  } else {
    Pair<SimtGemmArgs<bf16>> g; g.m[0] = g.m[1] = SimtGemmArgs<bf16>{nullptr, rows, (const bf16*)A_dev, (const bf16*)W_dev, out_dev, N, K};
    gemm_simt_kernel<bf16><<<grid, 256>>>(g);
  }
  return cudaDeviceSynchronize() == cudaSuccess ? TANDEM_OK : TANDEM_ECUDA;
}

int tandem_test_gemm_time(int32_t rows, int32_t N, int32_t K, int32_t iters, int32_t ring_kb, int32_t splits, int32_t flags, float* ms_per_launch) {
  if (rows <= 0 || N <= 0 || K <= 0 || iters <= 0 || !ms_per_launch) return TANDEM_EINVAL;
  TcGemmTune t; t.ring_kb = ring_kb; t.splits = splits; t.pdl = (flags & 2) != 0; t.pair = (flags & 4) ? 1 : 0;
  return tc_gemm_time(rows, N, K, iters, t, (flags & 1) ? kTcEpiSwiGLU : kTcEpiPartial, ms_per_launch);
}

int tandem_test_set_option(tandem_handle* h, const char* name, int32_t value) {
  if (!h || !name) return TANDEM_EINVAL;
  const std::string n(name);
  auto in = [&](int lo, int hi) { return value >= lo && value <= hi; };
  if (n == "pdl" && in(0, 1)) h->use_pdl = value != 0;
  else if (n == "attn_ctas_per_sm" && in(1, 2)) h->attn_ctas_per_sm = value;
  else if (n == "gemm_ring_kb" && in(0, 200)) h->gemm_ring_kb = value;
  else if (n == "fused_sampler" && in(0, 1)) h->fused_sampler = value != 0;
  else if (n == "gateup_streamk" && in(0, 1)) h->gateup_streamk = value != 0;
  else if (n == "attn_min_chunk" && (value == 0 || (value >= 64 && value % 64 == 0))) h->attn_min_chunk = value;
  else if (n == "skip_class" && in(-1, TANDEM_KC_NUM - 1)) h->skip_class = value;
  else if (n == "dual_forward" && in(0, 1)) h->dual_forward = value != 0;
  else if (n == "attn_prefill_tc" && in(0, 1)) h->attn_prefill_tc = value != 0;
  else if (n == "profile_catchup_attention" && in(0, 1)) h->profile_catchup_attn = value != 0;
  else return fail(h, TANDEM_EINVAL, "unknown option or value out of range: " + n);
  CU(h, cudaDeviceSynchronize());
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; h->gkey.valid = false; }
  return TANDEM_OK;
}

int tandem_test_set_page_order(tandem_handle* h, uint64_t seed) {
  if (!h) return TANDEM_EINVAL;
  h->page_order_seed = seed;
  return TANDEM_OK;
}

}  // extern "C"
