"""B200-native batched time-domain Gaussian log-likelihood (arxiv 2603.06010 hot path).

The public calls mirror the C ABI of include/tdlike.h (td_create, td_loglike_batch,
td_inner_batch, td_destroy, ...); see paper_2603_06010_b200.binding.  Importing this package
does not load the CUDA library; the first call into the binding does, and fails loudly if
the library is missing.
"""
__version__ = "0.1.0"
