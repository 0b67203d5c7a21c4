"""paper_2606_15650_b200 -- B200-native (sm_100a) hot path of AnonShield's pseudonymization pipeline.

The product is the C-ABI library `libanonshield.so` (csrc/, declared in include/anonshield.h); this package
is its thin Python binding.  See DESIGN.md.
"""
from .binding import (AnonError, Cache, Context, ModelDesc, Regex, Weights, anon_ctx_set_regex, anon_merge_spans, anon_regex_scan, anon_attention, anon_attention_local, anon_decode_spans, anon_decode_spans_static,  # noqa: F401
                      anon_gather_spans, anon_gemm_bf16, anon_hmac_spans, anon_splice_records, anon_ner_forward, anon_pipeline_host,
                      anon_pseudonymize, anon_workspace_bytes, anon_microbench, anon_gemm_bf16_fold, anon_gemm_bf16_fold_res, lib)
from .binding import OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CAPACITY, ERR_KEY_MISMATCH, ERR_CUDA, ERR_OOM  # noqa: F401
