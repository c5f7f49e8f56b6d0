"""paper_2606_15652_b200 -- B200 (sm_100a) hot path of MosaicQuant / ZipperEngine.

The product is the C-ABI library `libmq.so` (include/mq.h, sources in csrc/); this package is
its thin Python binding with the same entry-point names.  No CPU fallback exists.
"""
from .binding import (  # noqa: F401
    MQ_BF16,
    MQ_F16,
    EXPORTS,
    LIB_PATH,
    MqError,
    Weights,
    lib,
    mq_gemm,
    mq_gemm_a8,
    mq_gemm_group,
    mq_gemm_group_workspace_bytes,
    mq_gemm_naive,
    mq_gemm_naive_scratch_bytes,
    mq_gemm_workspace_bytes,
    mq_last_launch_count,
    mq_linear,
    mq_linear_host,
    mq_linear_host_staging_bytes,
    mq_linear_workspace_bytes,
    mq_pack_prequantized,
    mq_pack_weights,
    mq_pack_weights_device,
    mq_probe_int8_peak,
    mq_qact_bytes,
    mq_quantize_act,
    mq_quantize_act8,
    mq_quantize_act_group,
    mq_set_option,
    mq_unpack_act,
    new_workspace,
    status_string,
)
