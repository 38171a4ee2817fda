"""paper_2607_02945_b200 -- Python binding of liboptimus_b200 (sm_100a).

One kernel launch per horizontally fused op group (Optimus, arxiv/paper_2607_02945,
PAPER.md:148 group fusion).  The binding only marshals arguments: every step of
the hot path runs in the CUDA kernels behind the C ABI (include/optimus_b200.h).
There is no CPU fallback: importing fails loudly if the shared library is missing
and cannot be built.
"""
from .binding import (  # noqa: F401
    OPT_F32, OPT_BF16,
    OPT_ACT_NONE, OPT_ACT_RELU, OPT_ACT_TANH, OPT_ACT_SIGMOID,
    OPT_PW_COPY, OPT_PW_RELU, OPT_PW_TANH, OPT_PW_SIGMOID,
    OPT_PW_CLAMP, OPT_PW_NAN_TO_NUM, OPT_PW_SUB, OPT_PW_DIV, OPT_PW_MUL, OPT_PW_QUANT_E4M3, OPT_PW_DEQUANT_E4M3, OPT_PW_RELU_BWD, OPT_PW_TANH_BWD, OPT_PW_SIGMOID_BWD,
    OPT_LAYOUT_X_TRANSPOSED, OPT_LAYOUT_W_TRANSPOSED,
    OPT_OK, OPT_ERR_INVALID_ARG, OPT_ERR_UNSUPPORTED, OPT_ERR_ALIGNMENT, OPT_ERR_ALIAS, OPT_ERR_CUDA,
    OPT_ERR_NO_DEVICE,
    OptError, Plan, lib, lib_path,
    opt_linear_member, opt_linear_options, opt_linear2_member, opt_ln_linear2_member, opt_layernorm_member, opt_layernorm_bwd_member, opt_bias_grad_member, opt_chunk, opt_host_copy,
    opt_linear_plan_create, opt_linear_plan_create_ex, opt_linear2_plan_create, opt_ln_linear2_plan_create, opt_layernorm_plan_create, opt_layernorm_bwd_plan_create, opt_bias_grad_plan_create,
    opt_pointwise_plan_create, opt_bias_grad_noalloc, OPT_NOALLOC_BIAS_GRAD_MAX_N,
    opt_plan_launch, opt_plan_launch_host, opt_plan_info, opt_plan_destroy,
    opt_last_error, opt_launch_count, opt_version,
    linear_member, linear2_member, ln_linear2_member, layernorm_member, layernorm_bwd_member, bias_grad_member, chunk, split_cat_chunks,
)
