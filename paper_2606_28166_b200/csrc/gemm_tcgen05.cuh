// placeholder, replaced below
#pragma once
#include "common.cuh"
namespace tandem {
struct TcGemmPlans;
inline TcGemmPlans* tc_gemm_create() { return nullptr; }
inline void tc_gemm_destroy(TcGemmPlans*) {}
inline void tc_gemm_invalidate(TcGemmPlans*, int) {}
inline int tc_gemm_launch(TcGemmPlans*, int, int, int, const void*, const void*, int, int, float*, const int32_t*, int, int*, size_t*, cudaStream_t) { return -3; }
inline int tc_gemm_test(int, int, int, const void*, const void*, float*) { return -3; }
}
