// Senior-masked GRPO objective, forward only - SURVEY.md section 8(f) NEXT-3.
// PAPER.md L69-71 (section 3.4, Eq. 1), Table 3 (L277-292: clip 0.2, G = 8, group-relative std-normalised advantages, junior-token
// loss weight 0), Alg. 1 lines 19-21 (L370-376); reading R19 in DESIGN.md section 3 for what the paper leaves to Shao et al. 2024.
// Consumes what the rollout returns (owner flags, senior log-probs, lengths) and what tandem_score returns for the updated policy.
#pragma once
#include "common.cuh"

namespace tandem {

struct GrpoArgs {
  int n_seqs, group, stride;
  const float* rewards; const int32_t* len; const uint8_t* owner;
  const float* logp_new; const float* logp_old; const float* logp_ref;
  float clip_eps, kl_beta, adv_eps;
  float* advantages; float* token_obj; float* seq_obj;
  float* result;     // [8]: {loss, clip fraction, senior positions, live rollouts} then four integer scratch words, zero at launch
};

// One CTA per rollout i: A_i from its group's rewards, then J_i = mean over its senior positions of
// min(rho A, clip(rho, 1 - eps, 1 + eps) A) - beta k, rho = exp(new - old), k = exp(ref - new) - (ref - new) - 1.
template <int NT>
__global__ void __launch_bounds__(NT) grpo_seq_kernel(const __grid_constant__ GrpoArgs a) {
  __shared__ float red[32];
  const int i = blockIdx.x;
  const int g0 = (i / a.group) * a.group;
  // group statistics in double: G values, every CTA of the group computes the same numbers in the same order
  double mean = 0.0;
  for (int k = 0; k < a.group; ++k) mean += (double)a.rewards[g0 + k];
  mean /= (double)a.group;
  double var = 0.0;
  for (int k = 0; k < a.group; ++k) { const double d = (double)a.rewards[g0 + k] - mean; var += d * d; }
  var /= (double)a.group;
  const float A = (float)(((double)a.rewards[i] - mean) / (sqrt(var) + (double)a.adv_eps));
  const int n = min(a.len[i], a.stride);
  const size_t row = (size_t)i * a.stride;
  const float lo_c = 1.f - a.clip_eps, hi_c = 1.f + a.clip_eps;
  float acc = 0.f, cnt = 0.f, clipped = 0.f;
  for (int t = threadIdx.x; t < a.stride; t += NT) {
    float s = 0.f;
    if (t < n && a.owner[row + t] == 0) {
      const float ln = a.logp_new[row + t];
      const float rho = expf(ln - a.logp_old[row + t]);
      const float rc = fminf(fmaxf(rho, lo_c), hi_c);
      s = fminf(rho * A, rc * A);
      if (rc * A < rho * A) clipped += 1.f;   // the clipped branch is the one min() takes: the position whose gradient is cut (R19)
      if (a.kl_beta != 0.f && a.logp_ref) {
        const float d = a.logp_ref[row + t] - ln;
        s -= a.kl_beta * (expf(d) - d - 1.f);
      }
      acc += s;
      cnt += 1.f;
    }
    if (a.token_obj) a.token_obj[row + t] = s;
  }
  acc = block_sum<NT>(acc, red);
  cnt = block_sum<NT>(cnt, red);
  clipped = block_sum<NT>(clipped, red);
  __shared__ int s_last;
  int* scratch = reinterpret_cast<int*>(a.result) + 4;   // senior positions, clipped positions, live rollouts, arrivals
  if (threadIdx.x == 0) {
    a.advantages[i] = A;
    a.seq_obj[i] = cnt > 0.f ? acc / cnt : 0.f;
    atomicAdd(scratch + 0, (int)cnt);
    atomicAdd(scratch + 1, (int)clipped);
    atomicAdd(scratch + 2, cnt > 0.f ? 1 : 0);
    __threadfence();
    s_last = atomicAdd(scratch + 3, 1) == a.n_seqs - 1;
  }
  __syncthreads();
  if (!s_last) return;
  // the last rollout to finish reduces the per-rollout objectives in index order: loss = -(1/B) sum_i J_i
  __threadfence();
  float s = 0.f;
  for (int k = threadIdx.x; k < a.n_seqs; k += NT) s += __ldcg(a.seq_obj + k);
  s = block_sum<NT>(s, red);
  if (threadIdx.x == 0) {
    const int n_sen = __ldcg(scratch + 0), n_clip = __ldcg(scratch + 1), n_live = __ldcg(scratch + 2);
    a.result[0] = -s / (float)a.n_seqs;
    a.result[1] = n_sen > 0 ? (float)n_clip / (float)n_sen : 0.f;
    a.result[2] = (float)n_sen;
    a.result[3] = (float)n_live;
  }
}

}  // namespace tandem
