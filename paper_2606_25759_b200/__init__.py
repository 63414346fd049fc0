"""paper_2606_25759_b200 — B200-native (sm_100a) low-bit gradient-bucket aggregation.

The product is the C-ABI CUDA library libnf.so (include/nf.h, csrc/); `binding` marshals torch
CUDA tensors into its calls, `bucket.BucketBuffers` holds one bucket's device buffers.
"""
from . import binding  # noqa: F401
from .binding import (nf_route_bucket, nf_sign_pack, nf_sign_count_reduce, nf_fp32_reduce,  # noqa: F401
                      nf_health_stats, nf_aggregate_bucket, nf_aggregate_bucket_host,
                      nf_plan_bytes, nf_workspace_bytes, MODE_GBINARY, MODE_GTERNARY,
                      ROUTE_P, ROUTE_L, ROUTE_F, NfError)
from .bucket import BucketBuffers, ModelBuffers  # noqa: F401
