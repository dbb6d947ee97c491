"""paper_2606_01556_b200 -- B200 (sm_100a) TwinQuant dual-component 4-bit linear layer.

Thin Python binding over the C-ABI library libtwq.so (include/twq.h).  The binding only
marshals arguments (torch tensors -> device pointers, current stream); every step of the
hot path runs in the CUDA kernels under csrc/.  There is NO CPU or PyTorch fallback: if
the library is missing or the device is not sm_100 the calls raise.
"""
from .binding import (  # noqa: F401
    TwqError, lib_path, load_library, packed_bytes, workspace_bytes, pack_weights, quantize_act,
    dual_linear, dual_linear_x, dual_linear_noalloc, noalloc_max_workspace, workspace_bytes_x, pack_weights_q4lr, dual_linear_q4lr_x, algorithmic_bytes_q4lr, lowrank_group, last_launch_count, testing_set_plan_flags, testing_describe_plan, testing_set_trace_buffer, testing_measure_i8_tops, testing_cold_fill_us, plan_fused_cs, plan_decode_cs, plan_fused_tn_cap,
    PLAN_NO_SPLIT, PLAN_NO_PAIR, PLAN_NO_YSTAGE, PLAN_NO_ALIAS2, PLAN_NO_DECODE, OUT_BF16, OUT_FP16, OUT_FP32, PackedLayer, algorithmic_bytes, algorithmic_bytes_x, flops,
)
