"""sangam-b200: B200-native paged non-causal block attention + KV page write (arxiv/paper_2607_04206).

Thin Python binding over the C ABI in include/sangam.h.  Argument marshalling only: every step
of the path runs in the CUDA kernels of csrc/.  There is no CPU fallback -- if libsangam.so is
missing or a CUDA device is absent the calls raise.
"""
from .binding import (SangamError, Sangam, Scheduler, rope_table, load_library, exported_symbols, DECLARED_SYMBOLS,  # noqa: F401
                      DISPATCH_AUTO, DISPATCH_PREFILL, DISPATCH_DECODE, DISPATCH_GQA_PAIR,
                      confidence_sample_static, STATIC_SAMPLER_MAX_ROWS, STATIC_SAMPLER_MAX_PARTIALS)
