"""libjetlong: B200-native fused bifocal RoPE attention (Jet-Long, arxiv/paper_2607_07740)."""
from .binding import (BF16, FP32, JetlongError, jetlong_causal_decode, jetlong_causal_prefill,  # noqa: F401
                      jetlong_decode, jetlong_decode_paged, jetlong_decode_static, jetlong_decode_static_init, jetlong_group_size, jetlong_launch_count, jetlong_prefill,
                      jetlong_prefill_host, jetlong_prefill_prerotated, jetlong_prefill_unfused, jetlong_set_prefill_impl,
                      jetlong_set_prefill_precision,
                      jetlong_workspace_bytes, PRECISION_COMPENSATED, PRECISION_COMPENSATED_E5M2,
                      PRECISION_COMPENSATED_F16, PRECISION_FAST)
