// kernels.cuh - scheduler (S0), embedding+norm (S1,S2), GEMM epilogues (S2,S4,S6,S7) and the
// sample+switch+emit kernel (S8) of the tandem rollout engine. See DESIGN.md section 6.
#pragma once
#include "common.cuh"

namespace tandem {

// ============================================================================================ S0: scheduler
// One CTA, one thread per slot. For each model M: the sequences M owns get rows for the context positions M
// has not ingested yet (q_len = n_ctx - ing[M]; 1 = plain decode, >1 = catch-up / prompt prefill), capped by
// the row budget in slot order; pages are taken from M's free stack; row, emit and attention-item tables are
// written for the kernels downstream. PAPER.md L257 (per-step attention metadata: slot mappings, block tables,
// position indices) - here per model, since the two models are no longer in lock-step.
struct SchedArgs {
  SeqState st; PageTab pt[2]; GroupTab gt; StepTab tab[2]; StepIO io; DevStats* stats;
  const int32_t* tokens; int max_seqs, max_seq_len, max_pages, row_cap, tile_tok;
  int32_t* work_ctr; int n_work_ctr;   // dynamic-scheduling counters of the attention launches of this step
  int score;                           // teacher-forced dual scoring (tandem_score): both models ingest every sequence, every row reaches the LM head
  int no_parts;                        // tcgen05 scoring attention: every q-tile covers its whole causal KV range (no KV splits, no combine)
  int lockstep;                        // measurement (paper's engine): BOTH models ingest every token as it is emitted; only the owner samples
  int min_chunk;                       // smallest KV split (a function of the model shape only: kAttnMinChunk / kAttnMinChunkWide)
  int cascade;                         // share_prompt_pages = 2: the members of a group that a model serves in a step read the group's shared prompt pages ONCE (see below)
  int32_t* oom_flag;                   // mapped host word, set when a pool runs dry (the host reads it without synchronising)
};

__device__ __forceinline__ int block_excl_scan_1024(int v, int* total, int* wsum) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  if (w == 0) {
    int s = wsum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
    wsum[lane] = s;
  }
  __syncthreads();
  const int base = w > 0 ? wsum[w - 1] : 0;
  *total = wsum[31];
  __syncthreads();
  return base + x - v;
}

// last index s in [0, n) with cu[s] <= r, given cu non-decreasing and cu[n] > r
__device__ __forceinline__ int find_owner_slot(const int* cu, int n, int r) {
  int lo = 0, hi = n;  // invariant: cu[lo] <= r < cu[hi]
  while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (cu[mid] <= r) lo = mid; else hi = mid; }
  return lo;
}

__global__ void __launch_bounds__(1024) sched_kernel(SchedArgs a) {
  __shared__ int cu_rows[kMaxSlots + 1], cu_items[kMaxSlots + 1];
  __shared__ int sm_rows[kMaxSlots], sm_ing[kMaxSlots], sm_part0[kMaxSlots], sm_emit[kMaxSlots];
  // shared-prefix runs (cascade): per row-bearing index the run's group id (-1 = none) and the slot; per slot the shared length, the slot's
  // own item count, for a run's head its rows, and the index of the slot's first shared-prefix partial
  __shared__ short comp_eg[kMaxSlots], comp_slot[kMaxSlots];
  __shared__ unsigned short sm_ls[kMaxSlots], sm_oitems[kMaxSlots], sm_grows[kMaxSlots];
  __shared__ int sm_gp[kMaxSlots];
  __shared__ int wsum[32];
  const int s = threadIdx.x;
  const bool in_range = s < a.max_seqs;
  for (int i = threadIdx.x; i < a.n_work_ctr; i += blockDim.x) a.work_ctr[i] = 0;

  if (in_range) {  // defaults of the per-step outputs
    if (a.io.token) a.io.token[s] = -1;
    if (a.io.owner) a.io.owner[s] = 0;
    if (a.io.sen_logp) a.io.sen_logp[s] = 0.f;
    if (a.io.argmax) a.io.argmax[s] = -1;
  }
  const bool live = in_range && a.st.active[s] && !a.st.done[s];
  const int owner = live ? a.st.owner[s] : -1;
  const int nctx = live ? a.st.n_ctx[s] : 0;
  int resident_total;
  block_excl_scan_1024(live ? 1 : 0, &resident_total, wsum);
  const int nfeed = a.score ? nctx - 1 : nctx;   // scoring: the last token is only a target
  int fed[2] = {0, 0};
  int sched_rows_total = 0;   // thread 0 only

  for (int M = 0; M < 2; ++M) {
    const StepTab& tb = a.tab[M];
    const PageTab& pt = a.pt[M];
    const bool mine = (a.score || a.lockstep) ? live : owner == M;
    int ing = mine ? a.st.ing[M][s] : 0;
    // Prompt-page sharing: a member of a group that has not started with this model links the group's prompt pages if they are
    // ready, becomes the donor if nobody has started them, and otherwise waits (no rows this step) for the donor to finish.
    // g_state is read here, before the scans below; the donor publishes after them, so a step sees the state of its start.
    const int g = (mine && !a.score) ? a.st.grp[s] : -1;
    bool donor = false, waits = false;
    if (g >= 0 && ing == 0) {
      const int gs = a.gt.state[M][g];
      donor = gs == 1 && a.gt.donor[M][g] == s;
      if (gs == 2) {
        const int npg = a.gt.npg[g];
        for (int i = 0; i < npg; ++i) pt.bt[(size_t)s * a.max_pages + i] = a.gt.pages[M][(size_t)g * a.max_pages + i];
        pt.npages[s] = npg; pt.nshared[s] = npg;
        ing = npg * kPageTokens;
        a.st.ing[M][s] = ing;
        atomicAdd(&a.stats->shared_rows, (unsigned long long)ing);
      } else if (gs == 0) {
        if (atomicCAS(&a.gt.state[M][g], 0, 1) == 0) { a.gt.donor[M][g] = s; donor = true; } else waits = true;
      } else if (!donor) {
        waits = true;
      }
    } else if (g >= 0 && a.gt.state[M][g] == 1 && a.gt.donor[M][g] == s) {
      donor = true;   // a donor whose prefill is chunked over several steps
    }
    const int want = (mine && !waits) ? nfeed - ing : 0;
    int total_want;
    const int pre = block_excl_scan_1024(want, &total_want, wsum);
    int rows = min(want, max(0, a.row_cap - pre));   // tentative: the row budget in slot order
    // Pages for positions [ing, ing + rows), granted in slot order from the model's free stack. A sequence whose pages do not fit
    // any more is NOT scheduled this step (it stalls, nothing is written for it) and neither is any later slot that needs pages:
    // the pool never hands out a page twice and never points a block table at the dummy page. The host sees the stall through
    // DevStats::starved / the mapped flag: tandem_generate preempts a resident sequence, tandem_step reports a dead lock.
    {
      const int have = mine ? pt.npages[s] : 0;
      const int need = rows > 0 ? (ing + rows + kPageTokens - 1) / kPageTokens : 0;
      const int k = max(0, need - have);
      int total_k, total_g;
      const int kpre = block_excl_scan_1024(k, &total_k, wsum);
      const int free0 = *pt.free_top;                 // only this kernel and finalize_kernel (later in the stream) touch the stack
      const bool granted = kpre + k <= free0;
      block_excl_scan_1024(granted ? k : 0, &total_g, wsum);   // also orders every read of free_top before the write below
      if (k > 0 && granted) {
        for (int i = 0; i < k; ++i) pt.bt[(size_t)s * a.max_pages + have + i] = pt.free_pages[free0 - 1 - kpre - i];
        pt.npages[s] = need;
      }
      if (k > 0 && !granted) { rows = 0; atomicAdd(&a.stats->starved, 1ull); }
      if (threadIdx.x == 0 && total_k > 0) {
        *pt.free_top = free0 - total_g;
        if (total_g < total_k) { a.stats->err_oom = 1; if (a.oom_flag && *a.oom_flag < 1) *a.oom_flag = 1; }
      }
    }
    int n_rows;
    const int cu = block_excl_scan_1024(rows, &n_rows, wsum);
    const bool emits = !a.score && owner == M && mine && rows == want && want > 0;
    fed[M] = ing + rows;
    int n_emit;
    const int j = block_excl_scan_1024(emits ? 1 : 0, &n_emit, wsum);
    // attention items (S5): the rows of a sequence are cut into q-tiles of tile_tok tokens; q-tile t attends to the KV
    // range [0, ing + t0 + nt). For a sequence with at most kAttnSplitTiles q-tiles (decode, catch-ups) every q-tile is
    // also split along KV into chunks of attn_chunk(kv_len) positions whose partial (m, l, acc) are combined afterwards;
    // longer runs (prompt prefill) get their parallelism from the q-tiles and write their output directly.
    const int kv_len = ing + rows;
    const int n_qt = (rows + a.tile_tok - 1) / a.tile_tok;
    const int chunk = attn_chunk(kv_len, a.min_chunk);
    int n_sched;
    const int ridx = block_excl_scan_1024(rows > 0 ? 1 : 0, &n_sched, wsum);   // index among the slots that have rows in this model
    // Shared-prefix runs (share_prompt_pages = 2; the 8 rollouts of a GRPO group, hold the same prompt KV): the members of a group
    // that this model serves this step with all their rows past the shared prompt pages, and whose rows are neighbours in the row table, form
    // a run. The run's rows attend to the shared positions [0, Ls) TOGETHER - q-tiles over the run's rows, one partial per row - so those
    // pages are streamed once per run instead of once per member; every member's own items start at Ls, and the combine kernel merges the
    // shared partial with the member's own splits. Same sums up to the order of the softmax merge (the split point Ls).
    const int Ls_mine = (a.cascade && g >= 0) ? pt.nshared[s] * kPageTokens : 0;
    const bool elig = Ls_mine > 0 && rows > 0 && ing >= Ls_mine && n_qt <= kAttnSplitTiles && !a.no_parts;
    sm_rows[s] = rows;
    if (rows > 0) { comp_eg[ridx] = (short)(elig ? g : -1); comp_slot[ridx] = (short)s; }
    __syncthreads();
    const bool in_run = elig && ((ridx > 0 && comp_eg[ridx - 1] == g) || (ridx + 1 < n_sched && comp_eg[ridx + 1] == g));
    const bool head = in_run && !(ridx > 0 && comp_eg[ridx - 1] == g);
    int run_off = 0, run_rows = 0, head_slot = s;          // rows of the run before this member; head: rows of the whole run
    if (in_run) {
      for (int j2 = ridx - 1; j2 >= 0 && comp_eg[j2] == g; --j2) { run_off += sm_rows[comp_slot[j2]]; head_slot = comp_slot[j2]; }
      if (head) {
        int members = 0;
        for (int j2 = ridx; j2 < n_sched && comp_eg[j2] == g; ++j2) { run_rows += sm_rows[comp_slot[j2]]; ++members; }
        atomicAdd(&a.stats->kv_tokens_shared, (unsigned long long)(members - 1) * (unsigned long long)Ls_mine);
      }
    }
    const int Ls = in_run ? Ls_mine : 0;
    const int k_first = Ls / chunk;                          // own splits that lie wholly inside the shared prefix are not created
    const bool use_parts = rows > 0 && ((n_qt <= kAttnSplitTiles && kv_len > chunk && !a.no_parts) || in_run);
    int items = rows > 0 ? n_qt : 0, parts = 0;
    if (use_parts) {
      items = 0;
      for (int t = 0; t < n_qt; ++t) {
        const int t0 = t * a.tile_tok, nt = min(a.tile_tok, rows - t0);
        const int ns = (ing + t0 + nt + chunk - 1) / chunk - k_first;
        items += ns; parts += ns * nt;
      }
    }
    const int own_items = items, own_parts = parts;
    const int g_items = head ? (run_rows + a.tile_tok - 1) / a.tile_tok : 0;
    items += g_items; parts += head ? run_rows : 0;
    int n_items, n_parts, n_comb;
    const int icu = block_excl_scan_1024(items, &n_items, wsum);
    const int pcu = block_excl_scan_1024(parts, &n_parts, wsum);
    const int ccu = block_excl_scan_1024(use_parts ? rows : 0, &n_comb, wsum);

    cu_rows[s] = cu; cu_items[s] = icu;
    sm_ing[s] = ing; sm_part0[s] = use_parts ? pcu : -1; sm_emit[s] = emits ? j : -1;
    sm_ls[s] = (unsigned short)Ls; sm_oitems[s] = (unsigned short)own_items; sm_grows[s] = (unsigned short)(head ? run_rows : 0);
    sm_gp[s] = pcu + own_parts;                              // a head's shared-prefix partials follow its own
    if (s == 0) { cu_rows[kMaxSlots] = n_rows; cu_items[kMaxSlots] = n_items; }
    if (emits) tb.emit_slot[j] = s;
    __syncthreads();
    if (use_parts) {
      const int gp = in_run ? sm_gp[head_slot] + run_off : -1;
      int poff = 0;
      for (int t = 0; t < n_qt; ++t) {
        const int t0 = t * a.tile_tok, nt = min(a.tile_tok, rows - t0);
        const int ns = (ing + t0 + nt + chunk - 1) / chunk - k_first;
        for (int k = 0; k < nt; ++k) {
          tb.comb_row[ccu + t0 + k] = cu + t0 + k; tb.comb_part0[ccu + t0 + k] = pcu + poff + k;
          tb.comb_n[ccu + t0 + k] = ns; tb.comb_stride[ccu + t0 + k] = nt;
          tb.comb_gpart[ccu + t0 + k] = in_run ? gp + t0 + k : -1;
        }
        poff += ns * nt;
      }
    }
    if (rows > 0) a.st.ing[M][s] = ing + rows;  // commit: the forward below always runs
    if (donor && ing + rows >= a.gt.npg[g] * kPageTokens) {   // the shared prefix is stored after this step: hand its pages to the group
      const int npg = a.gt.npg[g];
      for (int i = 0; i < npg; ++i) a.gt.pages[M][(size_t)g * a.max_pages + i] = pt.bt[(size_t)s * a.max_pages + i];
      pt.nshared[s] = npg;
      a.gt.state[M][g] = 2;
    }
    __syncthreads();

    for (int r = threadIdx.x; r < n_rows; r += blockDim.x) {
      const int q = find_owner_slot(cu_rows, kMaxSlots, r);
      const int off = r - cu_rows[q];
      const int pos = sm_ing[q] + off;
      tb.row_slot[r] = q;
      tb.row_pos[r] = pos;
      tb.row_tok[r] = a.tokens[(size_t)q * a.max_seq_len + pos];
      tb.row_kvslot[r] = pt.bt[(size_t)q * a.max_pages + pos / kPageTokens] * kPageTokens + pos % kPageTokens;
      tb.row_emit[r] = a.score ? r : ((off == sm_rows[q] - 1) ? sm_emit[q] : -1);
    }
    for (int i = threadIdx.x; i < n_items; i += blockDim.x) {
      const int q = find_owner_slot(cu_items, kMaxSlots, i);
      const int off = i - cu_items[q];
      const int qrows = sm_rows[q], qkv = sm_ing[q] + qrows;
      if (off >= (int)sm_oitems[q]) {     // head of a shared-prefix run: q-tile t of the run's rows against the shared positions [0, Ls)
        const int t0 = (off - (int)sm_oitems[q]) * a.tile_tok, nt = min(a.tile_tok, (int)sm_grows[q] - t0);
        tb.item_row0[i] = cu_rows[q] + t0; tb.item_ntok[i] = nt;
        tb.item_kv0[i] = 0; tb.item_kv1[i] = (int)sm_ls[q];
        tb.item_part[i] = sm_gp[q] + t0;
      } else if (sm_part0[q] >= 0) {      // split sequence: walk its q-tiles to find (q-tile, split) number `off`
        const int ch = attn_chunk(qkv, a.min_chunk), ls = (int)sm_ls[q], kf = ls / ch;   // member of a run: its own items start at the shared length
        int rem = off, poff = 0, t0 = 0, nt = 0, ns = 0;
        for (;; t0 += a.tile_tok) {
          nt = min(a.tile_tok, qrows - t0);
          ns = (sm_ing[q] + t0 + nt + ch - 1) / ch - kf;
          if (rem < ns) break;
          rem -= ns; poff += ns * nt;
        }
        tb.item_row0[i] = cu_rows[q] + t0; tb.item_ntok[i] = nt;
        tb.item_kv0[i] = max((rem + kf) * ch, ls); tb.item_kv1[i] = min(sm_ing[q] + t0 + nt, (rem + kf + 1) * ch);
        tb.item_part[i] = sm_part0[q] + poff + rem * nt;
      } else {                            // q-tile `off`, whole causal range, written directly
        const int t0 = off * a.tile_tok, nt = min(a.tile_tok, qrows - t0);
        tb.item_row0[i] = cu_rows[q] + t0; tb.item_ntok[i] = nt;
        tb.item_kv0[i] = 0; tb.item_kv1[i] = sm_ing[q] + t0 + nt;
        tb.item_part[i] = -1;
      }
    }
    if (threadIdx.x == 0) {
      sched_rows_total += n_rows;
      tb.counts[C_ROWS] = n_rows; tb.counts[C_SCHED] = n_sched; tb.counts[C_EMIT] = a.score ? n_rows : n_emit;
      tb.counts[C_ITEMS] = n_items; tb.counts[C_COMB] = n_comb; tb.counts[C_PARTS] = n_parts;
      a.stats->rows[M] += (unsigned long long)n_rows;
      a.stats->catchup_rows += (unsigned long long)(n_rows - n_sched);
      a.stats->tokens_emitted += (unsigned long long)n_emit;
      if (n_rows > 0) a.stats->model_steps += 1ull;
    }
    // algorithmic KV tokens read this step: each scheduled sequence's owner reads its context once
    int kv_total;
    block_excl_scan_1024(rows > 0 ? ing + rows : 0, &kv_total, wsum);
    if (threadIdx.x == 0) a.stats->kv_tokens_read += (unsigned long long)kv_total;
    __syncthreads();
  }
  if (a.score && live && fed[0] >= nfeed && fed[1] >= nfeed) a.st.done[s] = 1;   // both models have seen the whole stream after this step
  if (threadIdx.x == 0) {
    a.stats->steps += 1ull;
    a.stats->peak_resident = max(a.stats->peak_resident, resident_total);
    // live sequences, not a single row scheduled, and pages were refused: no step can make progress any more without the host
    if (resident_total > 0 && sched_rows_total == 0 && a.stats->err_oom && a.oom_flag) *a.oom_flag = 2;
  }
}

// ============================================================================================ admission
struct AdmitArgs {
  SeqState st; PageTab pt[2]; GroupTab gt; int32_t* tokens; int max_seq_len;
  const int32_t* stage_tokens; const long long* stage_off; const int32_t* slots; const int32_t* seq_ids; const int32_t* max_new;
  const int32_t* grp; const int32_t* grp_members;   // per admitted sequence: its group (-1 = none); members of the group if it is the group's first, else 0
  int n; int start_owner; float p; unsigned long long seed; const float* u_switch; long long u_switch_stride;
};
__global__ void admit_kernel(AdmitArgs a) {
  const int i = blockIdx.x;
  if (i >= a.n) return;
  const int s = a.slots[i];
  const long long o0 = a.stage_off[i], o1 = a.stage_off[i + 1];
  for (long long k = o0 + threadIdx.x; k < o1; k += blockDim.x) a.tokens[(size_t)s * a.max_seq_len + (k - o0)] = a.stage_tokens[k];
  if (threadIdx.x == 0) {
    const int sid = a.seq_ids[i];
    int owner = a.start_owner;
    if (owner == 2) {  // DRAW: Alg. 1 line 6: senior iff u_switch[b,0] < p
      const float u = a.u_switch ? a.u_switch[(size_t)s * a.u_switch_stride] : u_switch_counter(a.seed, sid, 0);
      owner = (u < a.p) ? 0 : 1;
    }
    a.st.seq_id[s] = sid; a.st.prompt_len[s] = (int)(o1 - o0); a.st.n_ctx[s] = (int)(o1 - o0);
    a.st.ing[0][s] = 0; a.st.ing[1][s] = 0; a.st.cap_c[s] = 0; a.st.max_new[s] = a.max_new[i]; a.st.n_emit[s] = 0;
    a.st.owner[s] = (uint8_t)owner; a.st.done[s] = 0; a.st.active[s] = 1;
    a.pt[0].npages[s] = 0; a.pt[1].npages[s] = 0;
    a.pt[0].nshared[s] = 0; a.pt[1].nshared[s] = 0;
    const int g = a.grp ? a.grp[i] : -1;
    a.st.grp[s] = g;
    if (g >= 0 && a.grp_members[i] > 0) {   // first member: reset the group's entry
      a.gt.state[0][g] = 0; a.gt.state[1][g] = 0; a.gt.donor[0][g] = -1; a.gt.donor[1][g] = -1;
      a.gt.npg[g] = ((int)(o1 - o0) - 1) / kPageTokens;
      a.gt.ref[g] = a.grp_members[i];
    }
  }
}

// ============================================================================================ finalize
// After both models' samplers: release the pages of sequences that finished this step and count the rest.
struct FinalArgs { SeqState st; PageTab pt[2]; GroupTab gt; StepIO io; DevStats* stats; int32_t* n_active; int max_seqs, max_pages, pool_pages; };
__global__ void __launch_bounds__(1024) finalize_kernel(FinalArgs a) {
  __shared__ int wsum[32];
  const int s = threadIdx.x;
  bool live = false;
  if (s < a.max_seqs && a.st.active[s]) {
    if (a.st.done[s]) {
      for (int M = 0; M < 2; ++M) {   // the sequence's own pages; the leading nshared entries belong to its group
        const int n0 = a.pt[M].nshared[s], n = a.pt[M].npages[s] - n0;
        if (n > 0) {
          const int pos = atomicAdd(a.pt[M].free_top, n);
          for (int i = 0; i < n; ++i) {
            const int pg = a.pt[M].bt[(size_t)s * a.max_pages + n0 + i];
            if (pos + i < a.pool_pages) a.pt[M].free_pages[pos + i] = pg;   // after a pool exhaustion entries may name the dummy page 0: the handle then needs tandem_reset (tandem.h)
          }
        }
        a.pt[M].npages[s] = 0; a.pt[M].nshared[s] = 0;
      }
      const int g = a.st.grp[s];
      if (g >= 0 && atomicSub(&a.gt.ref[g], 1) == 1) {   // last member of its group: return the shared prompt pages
        for (int M = 0; M < 2; ++M) {
          if (a.gt.state[M][g] != 2) continue;
          const int n = a.gt.npg[g];
          const int pos = atomicAdd(a.pt[M].free_top, n);
          for (int i = 0; i < n; ++i)
            if (pos + i < a.pool_pages) a.pt[M].free_pages[pos + i] = a.gt.pages[M][(size_t)g * a.max_pages + i];
          a.gt.state[M][g] = 0;
        }
      }
      a.st.grp[s] = -1;
      a.st.active[s] = 0;
    } else {
      live = true;
    }
  }
  if (s < a.max_seqs && a.io.done) a.io.done[s] = a.st.done[s];
  int n_live;
  block_excl_scan_1024(live ? 1 : 0, &n_live, wsum);
  if (s == 0) {
    *a.n_active = n_live;
    if (a.io.n_active) *a.io.n_active = n_live;
    for (int M = 0; M < 2; ++M) {
      const int used = a.pool_pages - 1 - *a.pt[M].free_top;
      a.stats->peak_pages_used[M] = max(a.stats->peak_pages_used[M], used);
    }
  }
}

// ============================================================================================ S1+S2: embed + RMSNorm
// x[r,:] = E[token_r] (fp32 residual stream); u = x g / sqrt(mean x^2 + eps) -> act (GEMM A-operand dtype).
template <typename T> struct EmbedArgs { const int32_t* counts; const int32_t* row_tok; const T* E; const T* gain; float* x; T* act; int H; float eps; };
template <typename T, int NT>
__global__ void __launch_bounds__(NT) embed_norm_kernel(const __grid_constant__ Pair<EmbedArgs<T>> pp) {
  pdl_trigger(); pdl_wait();
  const EmbedArgs<T>& a = pp.m[blockIdx.y];
  const int32_t* __restrict__ counts = a.counts; const int32_t* __restrict__ row_tok = a.row_tok;
  const T* __restrict__ E = a.E; const T* __restrict__ gain = a.gain; float* __restrict__ x = a.x; T* __restrict__ act = a.act;
  const int H = a.H; const float eps = a.eps;
  __shared__ float red[32];
  const int n_rows = counts[C_ROWS];
  for (int r = blockIdx.x; r < n_rows; r += gridDim.x) {
    const T* e = E + (size_t)row_tok[r] * H;
    float ss = 0.f;
    for (int j = threadIdx.x; j < H; j += NT) { const float v = Elem<T>::ld(e + j); x[(size_t)r * H + j] = v; ss += v * v; }
    const float inv = rsqrtf(block_sum<NT>(ss, red) / (float)H + eps);
    for (int j = threadIdx.x; j < H; j += NT) Elem<T>::st(act + (size_t)r * H + j, Elem<T>::ld(e + j) * Elem<T>::ld(gain + j) * inv);
  }
}

// ============================================================================================ S6/S7: residual + RMSNorm
// x[r,:] += sum_s part[s][r,:] (ascending s); u = RMSNorm(x; gain) -> act. With out_map (last layer): only rows that emit
// are normalised (with the final-norm gain) and written compactly at their emit index (the LM head runs on those only).
// One CTA per row; every thread keeps its VPT float4 of the row in registers, and the loads of all splits are
// independent of each other, so a row costs ~one memory latency instead of n_split * H / NT of them.
template <typename T> struct ResNormArgs {
  const int32_t* counts; const float* part; int n_split; size_t split_stride; float* x; const T* gain; T* act; const int32_t* out_map; int H; float eps;
};
template <typename T, int NT, int VPT>
__global__ void __launch_bounds__(NT) residual_norm_kernel(const __grid_constant__ Pair<ResNormArgs<T>> pp) {
  pdl_trigger();
  const ResNormArgs<T>& a = pp.m[blockIdx.y];
  const int32_t* __restrict__ counts = a.counts; const float* __restrict__ part = a.part; const int n_split = a.n_split;
  const size_t split_stride = a.split_stride; float* __restrict__ x = a.x; const T* __restrict__ gain = a.gain; T* __restrict__ act = a.act;
  const int32_t* __restrict__ out_map = a.out_map; const int H = a.H; const float eps = a.eps;
  __shared__ float red[32];
  const int n_rows = counts[C_ROWS];
  const int H4 = H >> 2;
  // constants first (gains, scheduler tables): they do not depend on the predecessor kernel, so they load while it drains
  float4 gn[VPT];
#pragma unroll
  for (int i = 0; i < VPT; ++i) {
    const int j4 = threadIdx.x + i * NT;
    gn[i] = j4 < H4 ? ld4(gain + 4 * j4) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const int orow0 = (int)blockIdx.x < n_rows ? (out_map ? out_map[blockIdx.x] : (int)blockIdx.x) : -1;
  pdl_wait();
  for (int r = blockIdx.x; r < n_rows; r += gridDim.x) {
    float4 v[VPT];
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
      const int j4 = threadIdx.x + i * NT;
      v[i] = j4 < H4 ? ld4(x + (size_t)r * H + 4 * j4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll 8
    for (int s = 0; s < n_split; ++s) {
#pragma unroll
      for (int i = 0; i < VPT; ++i) {
        const int j4 = threadIdx.x + i * NT;
        if (j4 < H4) v[i] = add4(v[i], ld4(part + s * split_stride + (size_t)r * H + 4 * j4));
      }
    }
    float ss = 0.f;
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
      const int j4 = threadIdx.x + i * NT;
      if (j4 < H4) st4(x + (size_t)r * H + 4 * j4, v[i]);
      ss += v[i].x * v[i].x + v[i].y * v[i].y + v[i].z * v[i].z + v[i].w * v[i].w;
    }
    const int orow = r == (int)blockIdx.x ? orow0 : (out_map ? out_map[r] : r);
    const float inv = rsqrtf(block_sum<NT>(ss, red) / (float)H + eps);
    if (orow < 0) continue;
#pragma unroll
    for (int i = 0; i < VPT; ++i) {
      const int j4 = threadIdx.x + i * NT;
      if (j4 < H4) st4(act + (size_t)orow * H + 4 * j4, make_float4(v[i].x * gn[i].x * inv, v[i].y * gn[i].y * inv, v[i].z * gn[i].z * inv, v[i].w * gn[i].w * inv));
    }
  }
}

// ============================================================================================ S4: RoPE + KV append
// qkv[r, :] = sum_s part[s][r, :] is [q (nq*d) | k (nkv*d) | v (nkv*d)]. RoPE (half-split pairs (j, j+d/2), angle
// pos * theta^(-2j/d) from a table built in double at init) on q and k; q -> buffer of type QT (fp32 for the ALU attention
// kernel, bf16 for the tensor-core one), k and v -> model M's pages. Four pairs / four v elements per thread per step.
template <typename T, typename QT> struct RopeArgs {
  const int32_t* counts; const int32_t* row_pos; const int32_t* row_kvslot; const float* part; int n_split; size_t split_stride;
  const float2* cs_table; QT* q_out; T* kpool; T* vpool; int nq, nkv, d;
};
template <typename T, typename QT, int NT>
__global__ void __launch_bounds__(NT) rope_append_kernel(const __grid_constant__ Pair<RopeArgs<T, QT>> pp) {
  pdl_trigger(); pdl_wait();
  const RopeArgs<T, QT>& a = pp.m[blockIdx.y];
  const int32_t* __restrict__ counts = a.counts; const int32_t* __restrict__ row_pos = a.row_pos; const int32_t* __restrict__ row_kvslot = a.row_kvslot;
  const float* __restrict__ part = a.part; const int n_split = a.n_split; const size_t split_stride = a.split_stride;
  const float2* __restrict__ cs_table = a.cs_table; QT* __restrict__ q_out = a.q_out; T* __restrict__ kpool = a.kpool; T* __restrict__ vpool = a.vpool;
  const int nq = a.nq, nkv = a.nkv, d = a.d;
  const int n_rows = counts[C_ROWS];
  const int half = d >> 1, hq = half >> 2;                 // hq: groups of 4 pairs per head
  const int ld = (nq + 2 * nkv) * d;
  const int n_rot = (nq + nkv) * hq, n_v = nkv * (d >> 2);
  // four CTAs per row (blockIdx.x = 4 * row-lane + quarter): one item per thread at the 4B shape, so a row costs one memory latency
  const int quarter = blockIdx.x & 3;
  for (int r = blockIdx.x >> 2; r < n_rows; r += gridDim.x >> 2) {
    const int pos = row_pos[r];
    const int kvslot = row_kvslot[r];
    const int page = kvslot / kPageTokens, off = kvslot % kPageTokens;
    const float* src = part + (size_t)r * ld;
    for (int i = quarter * NT + threadIdx.x; i < n_rot + n_v; i += 4 * NT) {
      if (i < n_rot) {
        const int head = i / hq, j = (i - head * hq) << 2;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
#pragma unroll 4
        for (int s = 0; s < n_split; ++s) {
          a = add4(a, ld4(src + s * split_stride + head * d + j));
          b = add4(b, ld4(src + s * split_stride + head * d + j + half));
        }
        const float4 c01 = *reinterpret_cast<const float4*>(cs_table + (size_t)pos * half + j);       // (cos, sin) of pairs j, j+1
        const float4 c23 = *reinterpret_cast<const float4*>(cs_table + (size_t)pos * half + j + 2);
        const float4 ra = make_float4(a.x * c01.x - b.x * c01.y, a.y * c01.z - b.y * c01.w, a.z * c23.x - b.z * c23.y, a.w * c23.z - b.w * c23.w);
        const float4 rb = make_float4(b.x * c01.x + a.x * c01.y, b.y * c01.z + a.y * c01.w, b.z * c23.x + a.z * c23.y, b.w * c23.z + a.w * c23.w);
        if (head < nq) {
          st4(q_out + (size_t)r * nq * d + head * d + j, ra);
          st4(q_out + (size_t)r * nq * d + head * d + j + half, rb);
        } else {
          T* dst = kpool + (((size_t)page * nkv + (head - nq)) * kPageTokens + off) * d;
          st4(dst + j, ra); st4(dst + j + half, rb);
        }
      } else {
        const int e = (i - n_rot) << 2;                      // element index within [nkv * d)
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
        for (int s = 0; s < n_split; ++s) v = add4(v, ld4(src + s * split_stride + (nq + nkv) * d + e));
        const int kh = e / d;
        st4(vpool + (((size_t)page * nkv + kh) * kPageTokens + off) * d + (e - kh * d), v);
      }
    }
  }
}

// ============================================================================================ S7: SwiGLU
// gu[r, :] = [gate (I) | up (I)] summed over splits; out = silu(gate) * up, silu(a) = a / (1 + exp(-a)).
template <typename T> struct SwigluArgs { const int32_t* counts; const float* part; int n_split; size_t split_stride; T* out; int I; };
template <typename T, int NT>
__global__ void __launch_bounds__(NT) swiglu_kernel(const __grid_constant__ Pair<SwigluArgs<T>> pp) {
  pdl_trigger(); pdl_wait();
  const SwigluArgs<T>& a = pp.m[blockIdx.y];
  const int32_t* __restrict__ counts = a.counts; const float* __restrict__ part = a.part; const int n_split = a.n_split;
  const size_t split_stride = a.split_stride; T* __restrict__ out = a.out; const int I = a.I;
  const int n_rows = counts[C_ROWS];
  const int I4 = I >> 2;
  const size_t total = (size_t)n_rows * I4;
  for (size_t idx = (size_t)blockIdx.x * NT + threadIdx.x; idx < total; idx += (size_t)gridDim.x * NT) {
    const size_t r = idx / I4, j = (idx - r * I4) << 2;
    float4 g = make_float4(0.f, 0.f, 0.f, 0.f), u = g;
#pragma unroll 4
    for (int s = 0; s < n_split; ++s) {
      g = add4(g, ld4(part + s * split_stride + r * 2 * I + j));
      u = add4(u, ld4(part + s * split_stride + r * 2 * I + I + j));
    }
    st4(out + r * I + j, make_float4(g.x / (1.f + expf(-g.x)) * u.x, g.y / (1.f + expf(-g.y)) * u.y,
                                     g.z / (1.f + expf(-g.z)) * u.z, g.w / (1.f + expf(-g.w)) * u.w));
  }
}

// ============================================================================================ S8: sample + switch + emit
// n_chunk CTAs per emitting sequence of model M (slices of the vocabulary; the last to finish merges). logits row j (fp32, [n_emit, V]) -> token (forced | greedy argmax |
// Gumbel-max on position-addressed uniforms), log-prob under softmax(z/T'), authorship flag; then the rule of
// PAPER.md L61 / Alg. 1 lines 9-15 / L271: EOS or length => done; boundary = word_start[y]; cap counter; coin.
struct SampleArgs {
  SeqState st; StepTab tab; StepIO io; RuleParams rp; const float* logits; const uint8_t* word_start;
  int32_t* tokens; uint8_t* out_owner; float* out_logp; int vocab, max_seq_len, model;
  float* chunk_part;   // [max_seqs][n_chunk][6]: (max, sum, raw best value, raw best id, Gumbel best value, Gumbel best id) per vocabulary chunk
  int32_t* chunk_ctr;  // [max_seqs] arrival counters, zero between steps (the last arriver resets its own)
  int n_chunk;         // CTAs per row = gridDim.y
};

struct ArgBest { float v; int i; };
__device__ __forceinline__ ArgBest better(ArgBest a, ArgBest b) {  // larger value wins; ties: lower index
  return (b.v > a.v || (b.v == a.v && b.i < a.i)) ? b : a;
}

// The tail of S8 for one emitting sequence (slot s, token index t): append y, record owner flag and senior log-prob, then the rule of
// PAPER.md L61 / Alg. 1 lines 9-15 / L271: EOS or length => done; boundary = word_start[y]; cap counter; the coin decides a_{t+1}.
__device__ __forceinline__ void emit_token_and_switch(const SampleArgs& a, int s, int t, int sid, int y, float logp, int raw_id) {
  const int M = a.model;
  const int n = a.st.n_ctx[s];
  a.tokens[(size_t)s * a.max_seq_len + n] = y;
  a.out_owner[(size_t)s * a.max_seq_len + (t - 1)] = (uint8_t)M;
  a.out_logp[(size_t)s * a.max_seq_len + (t - 1)] = (M == 0) ? logp : 0.f;
  a.st.n_ctx[s] = n + 1;
  a.st.n_emit[s] = t;
  if (a.io.token) a.io.token[s] = y;
  if (a.io.owner) a.io.owner[s] = (uint8_t)M;
  if (a.io.sen_logp) a.io.sen_logp[s] = (M == 0) ? logp : 0.f;
  if (a.io.argmax) a.io.argmax[s] = raw_id;
  if ((a.rp.eos_id >= 0 && y == a.rp.eos_id) || t >= a.st.max_new[s]) { a.st.done[s] = 1; return; }
  // the rule: the coin after y_t decides the author of y_{t+1}
  const bool boundary = a.word_start[y] != 0;
  int c = boundary ? 0 : a.st.cap_c[s] + 1;
  int owner = M;
  if (boundary || (a.rp.cap_k > 0 && c >= a.rp.cap_k)) {
    const float u = a.io.u_switch ? a.io.u_switch[(size_t)s * a.io.u_switch_stride + t] : u_switch_counter(a.rp.seed, sid, t);
    const bool hit = u < a.rp.p;
    owner = (a.rp.switch_mode == 0) ? (hit ? 1 - M : M) : (hit ? 0 : 1);
    c = 0;
  }
  a.st.cap_c[s] = c;
  a.st.owner[s] = (uint8_t)owner;
}

// Nucleus (top-p) filtering, then the Gumbel argmax over the kept set (reading R10; off the fast path: a few passes over the
// L2-resident row by the CTA that merges it). Masses are fixed-point integers (exp(x - m) * 2^40), so every sum is exact and
// independent of the order of accumulation. Each id has a 24-bit depth T = floor(2^18 * min(log2e * (m - x), 64)), monotone in
// x. Level passes histogram the ids under the current prefix of T on its next 4 bits (16 bins of mass in registers, no atomics)
// and descend into the bin where the cumulative mass crosses top_p * total; from the second level on the same pass also
// gathers those ids into shared memory (an order-preserving 32-bit key of x, mass, id) and the descent stops once they fit.
// A bitwise search over the list finds the largest key k with mass{key >= k} >= target, i.e. the last kept probability. Ids
// above it are kept, ids equal to it by ascending id until the mass is reached. If the ids still do not fit after all 24 bits
// (a row of equal logits), the same search scans the row instead of the list. Last pass: the Gumbel argmax over the kept ids.
constexpr int kNucleusCap = 2048;
constexpr int kNucleusBins = 16;
template <int NT> struct NucleusSmem {
  unsigned long long ph[kNucleusBins][NT];   // a private histogram per thread: no atomics, no bank conflicts
  unsigned long long hist[kNucleusBins];
  unsigned long long cq[kNucleusCap];
  unsigned long long red[NT / 32];
  uint32_t ck[kNucleusCap];
  int cid[kNucleusCap];
  float redf[NT / 32];
  int redi[NT / 32];
  int n;
};
__device__ __forceinline__ uint32_t order_key(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key_value(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}
__device__ __forceinline__ uint32_t nucleus_depth(float d) { return (uint32_t)(fminf(d * 1.4426950408889634f, 63.99999f) * 262144.f); }
__device__ __forceinline__ unsigned long long nucleus_mass(float d) { return (unsigned long long)(expf(-d) * 1099511627776.f); }
template <int NT>
__device__ __forceinline__ unsigned long long block_sum_u64(unsigned long long v, unsigned long long* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  unsigned long long r = 0;
#pragma unroll
  for (int k = 0; k < NT / 32; ++k) r += red[k];
  return r;
}
// fn(z_v, v) over a row: 16-byte loads when the row allows, eight of them in flight per thread (one CTA reads the whole row
// out of L2, so the pass is bound by load latency)
template <int NT, typename F>
__device__ __forceinline__ void row_scan(const float* __restrict__ z, int V, F&& fn) {
  if ((V & 3) == 0 && (reinterpret_cast<uintptr_t>(z) & 15) == 0) {
    const float4* z4 = reinterpret_cast<const float4*>(z);
    const int n4 = V >> 2;
    constexpr int U = 8;
    int i = threadIdx.x;
    for (; i + (U - 1) * NT < n4; i += U * NT) {
      float4 q[U];
#pragma unroll
      for (int k = 0; k < U; ++k) q[k] = __ldg(z4 + i + k * NT);
#pragma unroll
      for (int k = 0; k < U; ++k) {
        const int v = 4 * (i + k * NT);
        fn(q[k].x, v); fn(q[k].y, v + 1); fn(q[k].z, v + 2); fn(q[k].w, v + 3);
      }
    }
    for (; i < n4; i += NT) {
      const float4 q = __ldg(z4 + i);
      fn(q.x, 4 * i); fn(q.y, 4 * i + 1); fn(q.z, 4 * i + 2); fn(q.w, 4 * i + 3);
    }
  } else {
    for (int v = threadIdx.x; v < V; v += NT) fn(__ldg(z + v), v);
  }
}
template <int NT>
__device__ int nucleus_gumbel_argmax(const float* __restrict__ z, int V, float invT, float m, float top_p, int top_k,
                                     const float* __restrict__ u_row, uint32_t k0, uint32_t k1, int t, int sid,
                                     NucleusSmem<NT>& S, uint8_t* keep_out = nullptr) {
  typedef unsigned long long u64;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool use_k = top_k > 0 && top_k < V, use_p = top_p < 1.f;
  uint32_t prefix = 0;
  u64 above = 0, target = 0;   // above: the mass of the ids shallower than the prefix (larger x)
  int lvl = 0;                 // the ids under the prefix: (T >> (24 - 4 lvl)) == prefix
  bool listed = false;
  // a filter keeps id v with key kx iff kx > key || (kx == key && v <= cut)
  uint32_t keyK = 0u, keyP = 0u;
  int cutK = V, cutP = V;
  auto append = [&](uint32_t k, u64 q, int v) {   // one counter increment for the lanes here
    const unsigned act = __activemask();
    const int leader = __ffs(act) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(&S.n, __popc(act));
    const int i = __shfl_sync(act, base, leader) + __popc(act & ((1u << lane) - 1u));
    if (i < kNucleusCap) { S.ck[i] = k; S.cq[i] = q; S.cid[i] = v; }
  };
  // c-th smallest id among the entries of `scan` with key == key
  auto tie_cut = [&](auto&& scan, uint32_t key, u64 c) {
    int lo = 0, hi = V - 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      u64 cnt = 0;
      scan([&](uint32_t k, u64, int id) { if (k == key && id <= mid) cnt += 1; });
      if (block_sum_u64<NT>(cnt, S.red) >= c) hi = mid; else lo = mid + 1;
    }
    return lo;
  };
  if (use_k) {
    // top-k (reading R18): the same descent on counts until the ids down to and including the bin of the k-th largest fit the list
    u64 cabove = 0;
    bool fits = false;
    while (lvl < 6 && !fits) {
      const int sh_pre = 24 - 4 * lvl, sh_bin = 20 - 4 * lvl;
#pragma unroll
      for (int k = 0; k < kNucleusBins; ++k) S.ph[k][threadIdx.x] = 0;
      row_scan<NT>(z, V, [&](float zv, int) {
        const uint32_t T = nucleus_depth(m - zv * invT);
        if ((T >> sh_pre) == prefix) S.ph[(T >> sh_bin) & (kNucleusBins - 1)][threadIdx.x] += 1;
      });
      __syncthreads();
      for (int k = w; k < kNucleusBins; k += NT / 32) {
        u64 hs = 0;
        for (int i = lane; i < NT; i += 32) hs += S.ph[k][i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) hs += __shfl_xor_sync(0xffffffffu, hs, o);
        if (lane == 0) S.hist[k] = hs;
      }
      __syncthreads();
      int bs = kNucleusBins - 1;
      bool found = false;
      for (int k = 0; k < kNucleusBins - 1; ++k) {
        if (!found) {
          if (cabove + S.hist[k] >= (u64)top_k) { bs = k; found = true; } else { cabove += S.hist[k]; }
        }
      }
      fits = cabove + S.hist[bs] <= (u64)kNucleusCap;
      prefix = (prefix << 4) | (uint32_t)bs;
      ++lvl;
      __syncthreads();
    }
    const int shk = 24 - 4 * lvl;
    if (threadIdx.x == 0) S.n = 0;
    __syncthreads();
    if (fits) {
      row_scan<NT>(z, V, [&](float zv, int v) {
        const float x = zv * invT, d = m - x;
        if ((nucleus_depth(d) >> shk) <= prefix) append(order_key(x), nucleus_mass(d), v);
      });
      __syncthreads();
      listed = true;
    }
    const int nk = listed ? S.n : 0;
    auto scan_k = [&](auto&& fn) {   // the list, or the whole row when even the deepest bin does not fit (a row of equal logits)
      if (listed) {
        for (int i = threadIdx.x; i < nk; i += NT) fn(S.ck[i], S.cq[i], S.cid[i]);
      } else {
        row_scan<NT>(z, V, [&](float zv, int v) { const float x = zv * invT; fn(order_key(x), nucleus_mass(m - x), v); });
      }
    };
    for (int bit = 31; bit >= 0; --bit) {   // the k-th largest key
      const uint32_t cand = keyK | (1u << bit);
      u64 c = 0;
      scan_k([&](uint32_t k, u64, int) { if (k >= cand) c += 1; });
      if (block_sum_u64<NT>(c, S.red) >= (u64)top_k) keyK = cand;
    }
    u64 gt = 0, eq = 0;
    scan_k([&](uint32_t k, u64, int) { if (k > keyK) gt += 1; if (k == keyK) eq += 1; });
    gt = block_sum_u64<NT>(gt, S.red);
    eq = block_sum_u64<NT>(eq, S.red);
    const u64 need = (u64)top_k - gt;
    if (need < eq) cutK = tie_cut(scan_k, keyK, need);
  }
  if (use_p && !use_k) {
    for (; lvl < 6; ++lvl) {
      if (threadIdx.x == 0) S.n = 0;
      __syncthreads();
      const int sh_pre = 24 - 4 * lvl, sh_bin = 20 - 4 * lvl;
      const bool gather = lvl > 0 || V <= kNucleusCap;
#pragma unroll
      for (int k = 0; k < kNucleusBins; ++k) S.ph[k][threadIdx.x] = 0;
      row_scan<NT>(z, V, [&](float zv, int v) {
        const float x = zv * invT, d = m - x;
        const uint32_t T = nucleus_depth(d);
        if ((T >> sh_pre) == prefix) {
          const int b = (T >> sh_bin) & (kNucleusBins - 1);
          const u64 q = nucleus_mass(d);
          S.ph[b][threadIdx.x] += q;
          if (gather) append(order_key(x), q, v);
        }
      });
      __syncthreads();
      for (int k = w; k < kNucleusBins; k += NT / 32) {   // bin k: the sum over all threads' private counters
        u64 hs = 0;
        for (int i = lane; i < NT; i += 32) hs += S.ph[k][i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) hs += __shfl_xor_sync(0xffffffffu, hs, o);
        if (lane == 0) S.hist[k] = hs;
      }
      __syncthreads();
      if (gather && S.n <= kNucleusCap) { listed = true; break; }
      u64 h[kNucleusBins];
#pragma unroll
      for (int k = 0; k < kNucleusBins; ++k) h[k] = S.hist[k];
      if (lvl == 0) {
        u64 total = 0;
#pragma unroll
        for (int k = 0; k < kNucleusBins; ++k) total += h[k];
        target = __double2ull_ru((double)top_p * (double)total);
        if (target < 1) target = 1;
      }
      int bs = kNucleusBins - 1;
      bool found = false;
#pragma unroll
      for (int k = 0; k < kNucleusBins - 1; ++k) {
        if (!found) {
          if (above + h[k] >= target) { bs = k; found = true; } else { above += h[k]; }
        }
      }
      prefix = (prefix << 4) | (uint32_t)bs;
      __syncthreads();
    }
  }
  if (use_p) {
    const int sh = 24 - 4 * lvl;
    const int n = listed ? S.n : 0;
    // fn(key, mass, id) over the candidates: the survivors of top-k, else the ids of the threshold bin
    auto scan = [&](auto&& fn) {
      if (listed) {
        for (int i = threadIdx.x; i < n; i += NT) {
          const uint32_t k = S.ck[i]; const int id = S.cid[i];
          if (!use_k || k > keyK || (k == keyK && id <= cutK)) fn(k, S.cq[i], id);
        }
      } else {
        row_scan<NT>(z, V, [&](float zv, int v) {
          const float x = zv * invT, d = m - x;
          const uint32_t k = order_key(x);
          if (use_k ? (k > keyK || (k == keyK && v <= cutK)) : ((nucleus_depth(d) >> sh) == prefix)) fn(k, nucleus_mass(d), v);
        });
      }
    };
    if (use_k || lvl == 0) {   // no level pass fixed the target: top-p renormalises over the top-k survivors / a short row sits in the list
      u64 tot = 0;
      scan([&](uint32_t, u64 q, int) { tot += q; });
      target = __double2ull_ru((double)top_p * (double)block_sum_u64<NT>(tot, S.red));
      if (target < 1) target = 1;
      above = 0;
    }
    for (int bit = 31; bit >= 0; --bit) {
      const uint32_t cand = keyP | (1u << bit);
      u64 f = 0;
      scan([&](uint32_t k, u64 q, int) { if (k >= cand) f += q; });
      if (above + block_sum_u64<NT>(f, S.red) >= target) keyP = cand;
    }
    u64 fs = 0, nt = 0;
    scan([&](uint32_t k, u64 q, int) { if (k > keyP) fs += q; if (k == keyP) nt += 1; });
    const u64 above_strict = above + block_sum_u64<NT>(fs, S.red);
    const u64 n_ties = block_sum_u64<NT>(nt, S.red);
    if (n_ties > 1) {
      const u64 q = nucleus_mass(m - key_value(keyP));
      u64 c = q ? (target - above_strict + q - 1) / q : n_ties;
      if (c < 1) c = 1;
      if (c < n_ties) cutP = tie_cut(scan, keyP, c);
    }
  }
  // the Gumbel argmax over the kept ids (Philox blocks of 4 ids, drawn only where an id is kept)
  ArgBest best = {-INFINITY, 0x7fffffff};
  const bool vec = (V & 3) == 0 && (reinterpret_cast<uintptr_t>(z) & 15) == 0;
#pragma unroll 2
  for (int b4 = threadIdx.x; b4 * 4 < V; b4 += NT) {
    float zz[4] = {0.f, 0.f, 0.f, 0.f};
    if (vec) { const float4 q = __ldg(reinterpret_cast<const float4*>(z) + b4); zz[0] = q.x; zz[1] = q.y; zz[2] = q.z; zz[3] = q.w; }
    else { for (int ww = 0; ww < 4 && b4 * 4 + ww < V; ++ww) zz[ww] = z[b4 * 4 + ww]; }
    uint32_t c[4] = {(uint32_t)b4, (uint32_t)t, (uint32_t)sid, 0u};
    bool drawn = u_row != nullptr;
#pragma unroll
    for (int ww = 0; ww < 4; ++ww) {
      const int v = b4 * 4 + ww;
      if (v >= V) break;
      const float x = zz[ww] * invT;
      const uint32_t kx = order_key(x);
      const bool keep = (kx > keyK || (kx == keyK && v <= cutK)) && (kx > keyP || (kx == keyP && v <= cutP));
      if (keep_out) keep_out[v] = keep;
      if (keep) {
        if (!drawn) { philox4x32_10(c, k0, k1); drawn = true; }
        const float u = u_row ? u_row[v] : uniform_from_bits(c[ww]);
        best = better(best, ArgBest{x + gumbel_from_uniform(u), v});
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ArgBest o2 = {__shfl_xor_sync(0xffffffffu, best.v, o), __shfl_xor_sync(0xffffffffu, best.i, o)};
    best = better(best, o2);
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { S.redf[w] = best.v; S.redi[w] = best.i; }
  __syncthreads();
  best = ArgBest{S.redf[0], S.redi[0]};
  for (int k = 1; k < NT / 32; ++k) best = better(best, ArgBest{S.redf[k], S.redi[k]});
  return best.i;
}

// test hook: one row of logits through the nucleus search exactly as the sampler runs it (explicit uniforms)
template <int NT>
__global__ void __launch_bounds__(NT) test_nucleus_kernel(const float* z, int V, float temperature, float top_p, int top_k, const float* u, int32_t* token,
                                                          uint8_t* keep) {
  extern __shared__ __align__(16) unsigned char nucleus_smem[];
  NucleusSmem<NT>& S = *reinterpret_cast<NucleusSmem<NT>*>(nucleus_smem);
  const float invT = 1.f / temperature;
  float m = -INFINITY;
  for (int v = threadIdx.x; v < V; v += NT) m = fmaxf(m, z[v] * invT);
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) S.redf[threadIdx.x >> 5] = m;
  __syncthreads();
  for (int k = 0; k < NT / 32; ++k) m = fmaxf(m, S.redf[k]);
  __syncthreads();
  const int y = nucleus_gumbel_argmax<NT>(z, V, invT, m, top_p, top_k, u, 0u, 0u, 1, 0, S, keep);
  if (threadIdx.x == 0) *token = y;
}

template <int NT, bool NUCLEUS>
__global__ void __launch_bounds__(NT) sample_switch_emit_kernel(const __grid_constant__ Pair<SampleArgs> pp) {
  pdl_trigger(); pdl_wait();
  const SampleArgs& a = pp.m[blockIdx.z];
  __shared__ float s_m[NT / 32], s_s[NT / 32], s_bv[NT / 32], s_gv[NT / 32];
  __shared__ int s_bi[NT / 32], s_gi[NT / 32];
  const int j = blockIdx.x;
  if (j >= a.tab.counts[C_EMIT]) return;
  // the vocabulary is cut into n_chunk slices (multiples of 4 ids = whole Philox blocks), one CTA each
  const int n_chunk = a.n_chunk, ch = blockIdx.y;
  const int per = (((a.vocab + 3) / 4 + n_chunk - 1) / n_chunk) * 4;
  const int v_lo = ch * per, v_hi = min(a.vocab, v_lo + per);
  const int s = a.tab.emit_slot[j];
  const int V = a.vocab;
  const float* z = a.logits + (size_t)j * V;
  const int t = a.st.n_emit[s] + 1;            // index of the token being emitted, 1-based
  const int sid = a.st.seq_id[s];
  const bool greedy = !(a.rp.temperature > 0.f);
  const float invT = greedy ? 1.f : 1.f / a.rp.temperature;
  const float* u_row = a.io.u_sample ? a.io.u_sample + ((size_t)s * a.io.u_sample_stride + (t - 1)) * V : nullptr;

  if (a.io.dbg_logits) {  // debug: the owner's logits for this position
    float* dst = a.io.dbg_logits + (size_t)s * V;
    for (int v = v_lo + threadIdx.x; v < v_hi; v += NT) dst[v] = z[v];
  }
  // one pass: running (max, sum exp) of z*invT for the log-softmax, raw argmax, Gumbel-perturbed argmax
  float m = -INFINITY, sum = 0.f;
  ArgBest raw = {-INFINITY, 0x7fffffff}, gum = {-INFINITY, 0x7fffffff};
  const uint32_t k0 = (uint32_t)a.rp.seed, k1 = (uint32_t)(a.rp.seed >> 32);
  for (int b4 = v_lo / 4 + threadIdx.x; b4 * 4 < v_hi; b4 += NT) {
    uint32_t c[4] = {(uint32_t)b4, (uint32_t)t, (uint32_t)sid, 0u};
    if (!greedy && !u_row) philox4x32_10(c, k0, k1);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int v = b4 * 4 + w;
      if (v >= V) break;
      const float zv = z[v];
      const float x = zv * invT;
      if (x > m) { sum = sum * expf(m - x) + 1.f; m = x; } else { sum += expf(x - m); }
      raw = better(raw, ArgBest{zv, v});
      if (!greedy) {
        const float u = u_row ? u_row[v] : uniform_from_bits(c[w]);
        gum = better(gum, ArgBest{x + gumbel_from_uniform(u), v});
      }
    }
  }
  // warp then block reduction
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float m2 = __shfl_xor_sync(0xffffffffu, m, o), s2 = __shfl_xor_sync(0xffffffffu, sum, o);
    const float mn = fmaxf(m, m2);
    sum = (m == -INFINITY ? 0.f : sum * expf(m - mn)) + (m2 == -INFINITY ? 0.f : s2 * expf(m2 - mn));
    m = mn;
    ArgBest o1 = {__shfl_xor_sync(0xffffffffu, raw.v, o), __shfl_xor_sync(0xffffffffu, raw.i, o)};
    raw = better(raw, o1);
    ArgBest o2 = {__shfl_xor_sync(0xffffffffu, gum.v, o), __shfl_xor_sync(0xffffffffu, gum.i, o)};
    gum = better(gum, o2);
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { s_m[w] = m; s_s[w] = sum; s_bv[w] = raw.v; s_bi[w] = raw.i; s_gv[w] = gum.v; s_gi[w] = gum.i; }
  __syncthreads();
  const bool nucleus = NUCLEUS && !greedy && (a.rp.top_p < 1.f || (a.rp.top_k > 0 && a.rp.top_k < a.vocab));   // the whole CTA stays for the nucleus search, else thread 0 alone
  if (!nucleus && threadIdx.x != 0) return;
  bool last = true;
  if (threadIdx.x == 0) {
    for (int k = 1; k < NT / 32; ++k) {
      const float mn = fmaxf(m, s_m[k]);
      sum = (m == -INFINITY ? 0.f : sum * expf(m - mn)) + (s_m[k] == -INFINITY ? 0.f : s_s[k] * expf(s_m[k] - mn));
      m = mn;
      raw = better(raw, ArgBest{s_bv[k], s_bi[k]});
      gum = better(gum, ArgBest{s_gv[k], s_gi[k]});
    }
    if (n_chunk > 1) {
      // publish this slice; the CTA that arrives last merges all slices in slice order (deterministic) and applies the rule
      float* cp = a.chunk_part + ((size_t)j * n_chunk + ch) * 6;
      cp[0] = m; cp[1] = sum; cp[2] = raw.v; cp[3] = __int_as_float(raw.i); cp[4] = gum.v; cp[5] = __int_as_float(gum.i);
      __threadfence();
      last = atomicAdd(a.chunk_ctr + j, 1) == n_chunk - 1;
      if (last) {
        a.chunk_ctr[j] = 0;
        __threadfence();
        m = -INFINITY; sum = 0.f; raw = ArgBest{-INFINITY, 0x7fffffff}; gum = raw;
        for (int k = 0; k < n_chunk; ++k) {
          const float* q = a.chunk_part + ((size_t)j * n_chunk + k) * 6;
          const float mk = __ldcg(q), sk = __ldcg(q + 1);
          const float mn = fmaxf(m, mk);
          sum = (m == -INFINITY ? 0.f : sum * expf(m - mn)) + (mk == -INFINITY ? 0.f : sk * expf(mk - mn));
          m = mn;
          raw = better(raw, ArgBest{__ldcg(q + 2), __float_as_int(__ldcg(q + 3))});
          gum = better(gum, ArgBest{__ldcg(q + 4), __float_as_int(__ldcg(q + 5))});
        }
      }
    }
  }
  bool searched = false;
  if constexpr (NUCLEUS) {
   if (nucleus) {
    extern __shared__ __align__(16) unsigned char nucleus_smem[];   // sizeof(NucleusSmem<NT>) when top_p < 1, else none
    __shared__ float s_fin;
    __shared__ int s_last;
    if (threadIdx.x == 0) { s_last = last; s_fin = m; }
    __syncthreads();
    if (!s_last) return;
    const int yn = nucleus_gumbel_argmax<NT>(z, V, invT, s_fin, a.rp.top_p, a.rp.top_k, u_row, k0, k1, t, sid, *reinterpret_cast<NucleusSmem<NT>*>(nucleus_smem));
    if (threadIdx.x != 0) return;
    gum.i = yn;
    searched = true;
   }
  }
  if (!searched && !last) return;
  int y = greedy ? raw.i : gum.i;
  if ((unsigned)y >= (unsigned)V) y = 0;   // all logits non-finite (NaN weights): no id ever won a comparison - emit id 0 rather than index out of bounds
  if (a.io.forced_tokens) {
    const int f = a.io.forced_tokens[(size_t)s * a.io.forced_stride + (t - 1)];
    if (f >= 0 && f < V) y = f;   // an id outside the vocabulary is ignored (it would index the logits and the embedding out of bounds)
  }
  emit_token_and_switch(a, s, t, sid, y, z[y] * invT - (m + logf(sum)), raw.i);
}

// ============================================================================================ S8, fused path: merge + emit
// The LM head's epilogue (gemm_tcgen05.cuh, kTcEpiSample) left one SamplePart per (emitting row, 128-id weight tile): [row][tile][8]
// fp32. One warp per emitting row merges the tiles - each lane its tiles in ascending order (eight loads in flight), then a butterfly over the lanes: a fixed
// tree, and sample_part_merge is symmetric, so every lane ends with the same bits - and lane 0 applies the rule. The logits never
// reached HBM: 38 KB of partials per row instead of 608 KB written and read.
struct SampleMergeArgs { SampleArgs sa; const float* part; int n_tiles; int row_cap; };
template <int NT>
__global__ void __launch_bounds__(NT) sample_merge_emit_kernel(const __grid_constant__ Pair<SampleMergeArgs> pp) {
  pdl_trigger(); pdl_wait();
  const SampleMergeArgs& ma = pp.m[blockIdx.y];
  const SampleArgs& a = ma.sa;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j = blockIdx.x * (NT / 32) + warp;
  if (j >= a.tab.counts[C_EMIT]) return;
  const bool greedy = !(a.rp.temperature > 0.f);
  const float invT = greedy ? 1.f : 1.f / a.rp.temperature;
  SamplePart acc{-INFINITY, 0.f, -INFINITY, 0.f, 0x7fffffff, 0x7fffffff};
  const float4* row = reinterpret_cast<const float4*>(ma.part + (size_t)j * ma.n_tiles * 8);
  for (int t0 = lane; t0 < ma.n_tiles; t0 += 8 * 32) {
    float4 p0[8], p1[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int t = t0 + 32 * k;
      p0[k] = make_float4(-INFINITY, 0.f, __int_as_float(0x7fffffff), -INFINITY); p1[k] = make_float4(__int_as_float(0x7fffffff), 0.f, 0.f, 0.f);
      if (t < ma.n_tiles) { p0[k] = __ldcg(row + 2 * t); p1[k] = __ldcg(row + 2 * t + 1); }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k)
      sample_part_merge(acc, SamplePart{p0[k].x, p0[k].y, p0[k].w, p1[k].y, __float_as_int(p0[k].z), __float_as_int(p1[k].x)}, invT);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    SamplePart b;
    b.m = __shfl_xor_sync(0xffffffffu, acc.m, o); b.s = __shfl_xor_sync(0xffffffffu, acc.s, o);
    b.gv = __shfl_xor_sync(0xffffffffu, acc.gv, o); b.gz = __shfl_xor_sync(0xffffffffu, acc.gz, o);
    b.raw_id = __shfl_xor_sync(0xffffffffu, acc.raw_id, o); b.g_id = __shfl_xor_sync(0xffffffffu, acc.g_id, o);
    sample_part_merge(acc, b, invT);
  }
  if (lane != 0) return;
  const int s = a.tab.emit_slot[j];
  const int t = a.st.n_emit[s] + 1;
  int y = greedy ? acc.raw_id : acc.g_id;
  if ((unsigned)y >= (unsigned)a.vocab) y = 0;   // all logits non-finite: see sample_switch_emit_kernel
  const float zy = greedy ? acc.m : acc.gz;
  emit_token_and_switch(a, s, t, a.st.seq_id[s], y, zy * invT - (acc.m * invT + logf(acc.s)), acc.raw_id);
}

// ============================================================================================ dual scoring (NEXT-1)
// PAPER.md L126 / L134 (section 4.4.2), reading R17: row r of the step holds position pos of sequence slot q in BOTH models
// (the scheduler keeps them in lock-step while scoring); with y = the stream's token at pos + 1 and p = softmax(z / T'):
//   out_sen[q][pos+1] = log p_sen(y), out_jun[q][pos+1] = log p_jun(y), out_alpha[q][pos+1] = sum_v min(p_sen(v), p_jun(v)).
// One CTA per row, two passes over the two fp32 logit rows: (max, sum exp) of each, then the min-sum.
struct ScoreArgs {
  const int32_t* counts; const int32_t* row_slot; const int32_t* row_pos; const int32_t* tokens; int max_seq_len;
  const float* z_sen; const float* z_jun; int vocab; float invT;
  float* out_sen; float* out_jun; float* out_alpha;
};
template <int NT>
__global__ void __launch_bounds__(NT) score_kernel(const __grid_constant__ ScoreArgs a) {
  pdl_trigger(); pdl_wait();
  __shared__ float red[32];
  __shared__ float s_m[2][NT / 32], s_s[2][NT / 32];
  const int V = a.vocab;
  const float invT = a.invT;
  const int n_rows = a.counts[C_ROWS];
  for (int r = blockIdx.x; r < n_rows; r += gridDim.x) {
    const float* zs = a.z_sen + (size_t)r * V;
    const float* zj = a.z_jun + (size_t)r * V;
    float m[2] = {-INFINITY, -INFINITY}, sum[2] = {0.f, 0.f};
    auto upd = [&](int k, float x) { if (x > m[k]) { sum[k] = sum[k] * expf(m[k] - x) + 1.f; m[k] = x; } else { sum[k] += expf(x - m[k]); } };
    row_scan<NT>(zs, V, [&](float zv, int) { upd(0, zv * invT); });
    row_scan<NT>(zj, V, [&](float zv, int) { upd(1, zv * invT); });
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, m[k], o), s2 = __shfl_xor_sync(0xffffffffu, sum[k], o);
        const float mn = fmaxf(m[k], m2);
        sum[k] = (m[k] == -INFINITY ? 0.f : sum[k] * expf(m[k] - mn)) + (m2 == -INFINITY ? 0.f : s2 * expf(m2 - mn));
        m[k] = mn;
      }
      if (l == 0) { s_m[k][w] = m[k]; s_s[k][w] = sum[k]; }
    }
    __syncthreads();
    float lse[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {   // every thread merges the warps' results in the same order
      float mm = s_m[k][0], ss = s_s[k][0];
      for (int i = 1; i < NT / 32; ++i) {
        const float mn = fmaxf(mm, s_m[k][i]);
        ss = (mm == -INFINITY ? 0.f : ss * expf(mm - mn)) + (s_m[k][i] == -INFINITY ? 0.f : s_s[k][i] * expf(s_m[k][i] - mn));
        mm = mn;
      }
      lse[k] = mm + logf(ss);
    }
    float acc = 0.f;
    if ((V & 3) == 0 && ((reinterpret_cast<uintptr_t>(zs) | reinterpret_cast<uintptr_t>(zj)) & 15) == 0) {
      const float4* a4 = reinterpret_cast<const float4*>(zs);
      const float4* b4 = reinterpret_cast<const float4*>(zj);
#pragma unroll 4
      for (int i = threadIdx.x; i < (V >> 2); i += NT) {
        const float4 p = __ldg(a4 + i), q = __ldg(b4 + i);
        acc += fminf(expf(p.x * invT - lse[0]), expf(q.x * invT - lse[1])) + fminf(expf(p.y * invT - lse[0]), expf(q.y * invT - lse[1])) +
               fminf(expf(p.z * invT - lse[0]), expf(q.z * invT - lse[1])) + fminf(expf(p.w * invT - lse[0]), expf(q.w * invT - lse[1]));
      }
    } else {
      for (int v = threadIdx.x; v < V; v += NT) acc += fminf(expf(zs[v] * invT - lse[0]), expf(zj[v] * invT - lse[1]));
    }
    acc = block_sum<NT>(acc, red);
    if (threadIdx.x == 0) {
      const int q = a.row_slot[r], pos = a.row_pos[r];
      const int y = a.tokens[(size_t)q * a.max_seq_len + pos + 1];
      const size_t o = (size_t)q * a.max_seq_len + pos + 1;
      a.out_sen[o] = zs[y] * invT - lse[0];
      a.out_jun[o] = zj[y] * invT - lse[1];
      a.out_alpha[o] = acc;
    }
    __syncthreads();
  }
}

}  // namespace tandem
