"""B200-native denoising step for masked diffusion language models (TeDiServe's GPU hot path).

The product is libdlm.so (CUDA for sm_100a behind the C ABI of include/dlm.h); this package is its thin
ctypes binding.  Nothing here falls back to a CPU implementation.
"""
from .binding import (DLM_DRY_RUN, EPI_BF16, EPI_F32, EPI_RESID, EPI_SWIGLU, FEATURE_NAMES, KIND_CACHED, KIND_MIXED, KIND_REFRESH, LIB_PATH,  # noqa: F401
                      OPT_CUDA_GRAPH, OPT_DEBUG_DUMP, OPT_FLASH_ATTENTION, OPT_KERNEL_TIMING, OPT_PDL, OPT_SIMPLE_KERNELS, OPT_SKINNY_GEMM, OPT_PAIR_GEMM, OPT_TC_ATTENTION, OPT_FUSE_ROPE, OPT_TRACE, OPT_TCT_MIN_ITEMS, OPT_LAYER_KERNEL, OPT_LAYER_KERNEL_PHASE_TS, DTYPE_BF16_PRECISE, PATH_LAYER_KERNEL,
                      PATH_ATTN_FLASH, PATH_ATTN_PLAIN, PATH_ATTN_TC, PATH_ATTN_TCT, PATH_GEMM_PAIR, PATH_GEMM_PLAIN, PATH_GEMM_SKINNY, PATH_GEMM_TC, PATH_GRAPH_REPLAY, PATH_ROPE_FUSED, DlmError, Engine,
                      StepResult, exported_symbols, lib, op_attention_bf16, op_gemm_bf16, op_gemm_pair_bf16, op_gemm_pair_plan, op_gemm_plain_bf16, op_gemm_skinny_bf16,
                      op_lmhead_bf16, op_lmhead_static_bf16, op_lmhead_unmask_bf16,
                      LMHEAD_STATIC_MAX_ROWS, LMHEAD_STATIC_SCRATCH_BYTES)
from . import binding  # noqa: F401
