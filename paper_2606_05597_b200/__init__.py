"""B200-native fused AsyncWebRL token loss (decoupled-PPO / multi-step GRPO, Eq. 1)
and its gradient over the LM-head vocabulary: hand-written sm_100a CUDA kernels behind the C ABI
of include/awr.h (libawr.so), plus this thin torch-tensor binding.  No CPU fallback exists."""
from ._abi import (AwrError, DTYPE_BF16, DTYPE_F32, ERRBIT_GROUP_OFF, ERRBIT_STEP_OFF,
                   ERRBIT_TARGET_RANGE, ERRBIT_TRAJ_OFF, FLAG_SAMPLE_STD, FLAG_SUCCESS_FILTER, FLAG_COUPLED, FLAG_SKIP_UNIFORM, KERNEL_AUTO,
                   KERNEL_CLUSTER, KERNEL_CLUSTER_RF, KERNEL_CLUSTER_RF4, KERNEL_CLUSTER_RFS, KERNEL_CLUSTER_RFS_LATE, KERNEL_GENERIC, KERNEL_HEAD_1CTA, KERNEL_HEAD_2CTA, KERNEL_HEAD_2CTA_STORED, KERNEL_HEAD_2CTA_E16, KERNEL_HEAD_2CTA_ROWREF, KERNEL_FWD_STREAM, NORM_CONST_K, NORM_PER_TRAJ, W_K_BY_V,
                   W_V_BY_K, STATIC_WS_BYTES, lib_path, load)
from .api import (HEAD_OPTIONAL_OUTPUTS, HeadLossCall, HostHeadLossCall, HostLossCall, LossCall, head_host_workspace_bytes, awr_gemm_bf16,
                  awr_loss_fwd_bwd_fused_head, head_launches_per_call, head_workspace_bytes, OPTIONAL_OUTPUTS, awr_group_advantage, awr_loss_fwd,
                  awr_loss_fwd_bwd, awr_loss_fwd_bwd_host, host_workspace_bytes,
                  launches_per_call, make_params, select_kernel, workspace_bytes,
                  StaticLossCall, awr_loss_fwd_bwd_static)
