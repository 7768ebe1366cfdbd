"""paper_2204_06633_b200 — B200-native generic time-domain LISA response (arXiv:2204.06633).

The product is liblr.so (csrc/, C ABI in include/lr.h).  This package is its thin Python binding and
nothing else (the seeded synthetic input generators live in the top-level `harness` package).  Importing the
binding does not load CUDA; the first call does, and fails loudly (`LrUnavailable`) if liblr.so has not been built.
"""
from .binding import (LR_AET, LR_CHAIN_NESTED, LR_CHAIN_SUM, LR_ECUDA, LR_EINVAL, LR_ENOMEM, LR_ERANGE,  # noqa: F401
                      LR_MAX_ORDER, LR_OK, LR_OPT_CHAIN, LR_OPT_CHANNELS, LR_OPT_T0, LR_OPT_TDI_GEN, LR_OPT_TDI_PATH, LR_OPT_TDI_PLAN_CACHE, LR_OPT_CHUNK_SAMPLES, LR_IP_CROSS, LR_IP_DIFF, LR_TDI_AUTO, LR_TDI_FIR3, LR_TDI_FIR4, LR_TDI_PER_SAMPLE, LR_XYZ,
                      LR_XYZ_AET, LrError, LrUnavailable, lr_create, lr_destroy, lr_eval_orbit, lr_get_margins, lr_get_option,
                      lr_launch_count, lr_plan_create, lr_plan_attach, lr_plan_release, lr_plan_bytes, lr_measure_fp64_peak, lr_get_span_halo, lr_inner_product, lr_inner_product_static, LR_ELIMIT, LR_IP_STATIC_MAX_BATCH, lr_gb_parameters, lr_fft_good_length, LR_OPT_FFT_LENGTH, LR_OPT_PROJ_PATH, LR_OPT_Y_PRECISION, LR_Y_PLAIN, LR_Y_EXTENDED, LR_INFO_TDI_PATH, LR_INFO_FIR_TAPS, LR_INFO_FIR_POWERS, LR_PROJ_AUTO, LR_PROJ_SINGLE, LR_PROJ_PAIR, lr_gb_waveform, lr_response_gb, lr_loglike_gb, LR_GB_NPAR, LR_GB_PAPER, LR_GB_CONFIG, lr_project, lr_response, lr_response_host, lr_response_span, lr_set_option,
                      lr_strerror, lr_tdi)
from .response import Response, gather_scalars, shard_templates, shard_time  # noqa: F401
