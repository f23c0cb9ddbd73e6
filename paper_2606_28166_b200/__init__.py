"""paper_2606_28166_b200 - B200-native tandem rollout (Tandem RLVR, arxiv/paper_2606_28166).

The product is the C-ABI library `libtandem.so` (include/tandem.h; hand-written sm_100a CUDA in csrc/).
This package is the thin Python binding over it: argument marshalling only, same names as the C calls.
PyTorch is used for device memory and streams. There is no CPU fallback: importing works anywhere (so
the symbol-export test can run without a GPU), but every compute call needs the library and a CUDA device.
"""
from .binding import (lib, lib_path, TandemConfig, TandemParams, Tandem, TandemError,
                      grpo_objective, grpo_objective_static, GRPO_STATIC_MAX_ROLLOUTS, tandem_test_uniforms, tandem_test_nucleus, tandem_test_philox, tandem_test_gemm, tandem_test_gemm_time,
                      SENIOR, JUNIOR, DRAW, TOGGLE, REDRAW, F32, BF16, GEMM_AUTO, GEMM_SIMT, GEMM_TCGEN05, ATTN_AUTO, ATTN_ALU, ATTN_MMA,
                      EXPORTED_SYMBOLS)
from .build import build

__all__ = ["lib", "lib_path", "TandemConfig", "TandemParams", "Tandem", "TandemError", "build",
           "grpo_objective", "grpo_objective_static", "GRPO_STATIC_MAX_ROLLOUTS", "tandem_test_uniforms", "tandem_test_nucleus", "tandem_test_philox", "tandem_test_gemm", "tandem_test_gemm_time",
           "SENIOR", "JUNIOR", "DRAW", "TOGGLE", "REDRAW", "F32", "BF16",
           "GEMM_AUTO", "GEMM_SIMT", "GEMM_TCGEN05", "ATTN_AUTO", "ATTN_ALU", "ATTN_MMA", "EXPORTED_SYMBOLS"]
