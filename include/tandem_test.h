/* tandem_test.h - measurement and unit-test hooks of libtandem.so. Not part of the product API (include/tandem.h): bench.py's
 * per-kernel roofline leg and the tests use them; a user of the library needs none of them. Same conventions as tandem.h. */
#ifndef TANDEM_TEST_H_
#define TANDEM_TEST_H_

#include "tandem.h"

#ifdef __cplusplus
extern "C" {
#endif

/* kernel classes of one step, for launch accounting and tandem_get_profile */
enum { TANDEM_KC_SCHED = 0, TANDEM_KC_EMBED, TANDEM_KC_GEMM_QKV, TANDEM_KC_ROPE_APPEND, TANDEM_KC_ATTENTION, TANDEM_KC_ATTN_COMBINE,
       TANDEM_KC_GEMM_O, TANDEM_KC_RESIDUAL_NORM, TANDEM_KC_GEMM_GATEUP, TANDEM_KC_SWIGLU, TANDEM_KC_GEMM_DOWN, TANDEM_KC_GEMM_LMHEAD,
       TANDEM_KC_SAMPLE, TANDEM_KC_FINALIZE, TANDEM_KC_SCORE, TANDEM_KC_ATTN_CATCHUP, TANDEM_KC_ATTN_EMPTY, TANDEM_KC_NUM };

/* Per-kernel timing mode (bench.py's roofline leg): while enabled, a step runs un-captured on the caller's stream, every kernel
 * bracketed by CUDA events, and the call returns after the step has finished. Results are unchanged. enable = 1 also zeroes
 * the accumulators. */
int tandem_set_profile(tandem_handle *h, int enable);
/* HOST out arrays of TANDEM_KC_NUM entries: accumulated device milliseconds and launch counts per kernel class. */
int tandem_get_profile(tandem_handle *h, double *ms, int64_t *launches);
const char *tandem_kernel_class_name(int kc);

/* A/B knob for measurements, by name; call before the first step (a captured step graph is dropped). Names: "pdl" (0/1, default 1),
 * "attn_ctas_per_sm" (1/2), "gemm_ring_kb" (0 = automatic), "fused_sampler" (0 = always materialise the logits and run the
 * separate sampler kernel; default 1: S8 in the LM head's epilogue when no filter / override / logits tap needs them), "profile_catchup_attention" (0/1: in profile mode launch the attention kernel a second time on the
 * catch-up items only - q_len > 1 - as class attention_catchup, and a third time with no item at all - class attention_empty, the
 * fixed cost of such a launch; results unchanged),  "gemm_pair" (-1 automatic, 0, 1), "score_nosplit" (0/1),
 * "score_chunk_grid" (1..16), "attn_prefill_tc" (0 = tandem_score runs its attention on the mma.sync kernel of the rollout; default 1:
 * the tcgen05 kernel over 128-row q-tiles, csrc/attention_tcgen05.cuh), "dual_forward" (1 = the paper's own engine for an on-box
 * comparison, PAPER.md L257 / SURVEY.md section 8(f)-1: BOTH models ingest every token in the step after it is emitted, so there is
 * no catch-up prefill and each model reads its whole KV cache every step; only the owner's row reaches the LM head and the sampler, so
 * tokens, owner flags and log-probs follow the same rule and the same random numbers; default 0 = owner split), "gateup_streamk" (0 = the
 * gate/up projection always runs on the one-tile-per-CTA kernel; default 1: decode-sized steps of a shape with at least one tile pair per
 * CTA use the persistent balanced kernel, csrc/gemm_streamk.cuh), "attn_min_chunk" (0 = by shape: 1024 KV positions per split for
 * models with >= 8 KV heads, else 256; or a multiple of 64), "skip_class" (-1 = none; a TANDEM_KC_* value: the launches of that
 * kernel class are left out of every step - the step's results are then garbage, its time less the full step's time is the class's
 * marginal cost inside the step graph, PDL overlap included; bench.py --skip-class). TANDEM_EINVAL for an unknown name or a value out of range. Every published number uses the defaults. */
int tandem_test_set_option(tandem_handle *h, const char *name, int32_t value);

/* Parity tests at realistic page numbers: seed != 0 makes tandem_reset (and so tandem_generate / tandem_score) hand the pages of each
 * pool out in a pseudo-random order (a seeded permutation of 1..pool-1) instead of ascending, so that short tests touch scattered,
 * high-numbered pages as a long-running engine does. 0 restores ascending order. Takes effect at the next reset. */
int tandem_test_set_page_order(tandem_handle *h, uint64_t seed);

/* ---- single kernels of the path, DEVICE pointers, synchronous ---- */

/* u[i] for i < n: the library's counter generator on stream `stream` (0 sample: v = i; 1 switch: t = i, v = 0). */
int tandem_test_uniforms(uint64_t seed, int32_t seq_id, int32_t t, int32_t stream, int32_t n, float *out_dev);
/* One row of fp32 logits [vocab] (DEVICE) through the sampler's top-k / top-p search with explicit uniforms u [vocab] (DEVICE):
 * token_dev <- the Gumbel argmax over the kept set, keep_dev [vocab] <- 1 where the id is kept (readings R10, R18). temperature > 0,
 * 0 < top_p <= 1, top_k <= 2048 (<= 0: off). */
int tandem_test_nucleus(int32_t vocab, float temperature, float top_p, int32_t top_k, const float *logits_dev, const float *u_dev, int32_t *token_dev,
                        uint8_t *keep_dev);
/* raw Philox-4x32-10 block, HOST in/out (runs on the device). */
int tandem_test_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* out[rows,N] (fp32) = A[rows,K] * W[N,K]^T with the selected GEMM implementation; dtype of A and W as given.
 * impl = 3: the tcgen05 kernel with its fused SwiGLU epilogue - W rows interleaved (2i = gate_i, 2i+1 = up_i), out is bf16
 * [rows, N/2] = silu(A gate_i) * (A up_i). impl = 4, 5: the same two kernels launched as CTA pairs (cta_group::2: two adjacent weight
 * tiles share one M = 256 MMA and each CTA loads half of the token rows). */
int tandem_test_gemm(int32_t dtype, int32_t impl, int32_t rows, int32_t N, int32_t K, const void *A_dev, const void *W_dev, float *out_dev);
/* Mean device milliseconds of `iters` back-to-back launches of the tcgen05 GEMM [rows,K] x [N,K]^T on synthetic bf16 data, each launch
 * on a different weight buffer (more than the L2 holds in total). ring_kb / splits = 0: the library's own choice. flags: bit 0 = fused
 * SwiGLU epilogue, bit 1 = programmatic dependent launch, bit 2 = CTA pairs. HOST out. */
int tandem_test_gemm_time(int32_t rows, int32_t N, int32_t K, int32_t iters, int32_t ring_kb, int32_t splits, int32_t flags, float *ms_per_launch);

#ifdef __cplusplus
}
#endif
#endif /* TANDEM_TEST_H_ */
