// gemm_simt.cuh - out[r, n] = sum_k A[r, k] W[n, k] on plain fp32 FMAs (S3, S6, S7, LM head of the fp32 config).
// tcgen05 has no fp32 input kind (tf32 keeps 10 mantissa bits), so configs[0] ("logits within 1e-4") runs here;
// the bf16 instantiation is the reference the tcgen05 kernel is unit-tested against and a debugging fallback.
// k is accumulated in ascending order by a single thread per output: results do not depend on the batch.
#pragma once
#include "common.cuh"

namespace tandem {

constexpr int kSimtTile = 32;

// grid: (ceil(N/32), row-tile lanes); each CTA walks row tiles r0 = blockIdx.y*32, += gridDim.y*32 while r0 < n_rows.
template <typename T> struct SimtGemmArgs { const int32_t* n_rows_ptr; int n_rows_fixed; const T* A; const T* W; float* out; int N, K; };
template <typename T>
__global__ void __launch_bounds__(256) gemm_simt_kernel(const __grid_constant__ Pair<SimtGemmArgs<T>> pp) {
  pdl_trigger(); pdl_wait();
  const SimtGemmArgs<T>& a = pp.m[blockIdx.z];
  const int32_t* __restrict__ n_rows_ptr = a.n_rows_ptr; const int n_rows_fixed = a.n_rows_fixed;
  const T* __restrict__ A = a.A; const T* __restrict__ W = a.W; float* __restrict__ out = a.out; const int N = a.N, K = a.K;
  __shared__ float As[kSimtTile][kSimtTile + 1];
  __shared__ float Ws[kSimtTile][kSimtTile + 1];
  const int n_rows = n_rows_ptr ? *n_rows_ptr : n_rows_fixed;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
  const int n0 = blockIdx.x * kSimtTile;
  for (int r0 = blockIdx.y * kSimtTile; r0 < n_rows; r0 += gridDim.y * kSimtTile) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k0 = 0; k0 < K; k0 += kSimtTile) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int rr = ty + 8 * i;
        const int k = k0 + tx;
        As[rr][tx] = (r0 + rr < n_rows && k < K) ? Elem<T>::ld(A + (size_t)(r0 + rr) * K + k) : 0.f;
        Ws[rr][tx] = (n0 + rr < N && k < K) ? Elem<T>::ld(W + (size_t)(n0 + rr) * K + k) : 0.f;
      }
      __syncthreads();
#pragma unroll
      for (int kk = 0; kk < kSimtTile; ++kk) {
        const float w = Ws[tx][kk];
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[i] = fmaf(As[ty + 8 * i][kk], w, acc[i]);
      }
      __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = r0 + ty + 8 * i, n = n0 + tx;
      if (r < n_rows && n < N) out[(size_t)r * N + n] = acc[i];
    }
  }
}

}  // namespace tandem
