"""The cases compute-sanitizer is run on (profiles/r2_sanitizer.md): every kernel family of the
library once, on inputs small enough for the tool's 10-100x slowdown.

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Not a pytest module (no test_ prefix): it only launches the kernels and checks that the error word
is clean; numerics are the parity tests' business."""
import os
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_2606_05597_b200 as A  # noqa: E402
from gen import workloads as W  # noqa: E402

DEV = "cuda:0"


def rows_case(w, kernel, backward=True, entropy=False):
    b = W.make_batch(w, seed=7, device=DEV, masked_frac=0.03)
    fn = A.awr_loss_fwd_bwd if backward else A.awr_loss_fwd
    want = A.OPTIONAL_OUTPUTS + (("token_entropy",) if entropy else ())
    out = fn(b["logits"], b["target_ids"], b["behave_lp"], b["prox_lp"], b["step_off"], b["traj_off"],
             b["group_off"], b["rewards"], want=want, **dict(b["params"], kernel=kernel, dual_clip_c=3.0))
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) == 0
    return float(out["loss"][0])


def head_case(kernel):
    w = W.workload(4, n_groups=4, group_size=4, n_tok=600, V=2056, hidden=128, lp_mode="drift")
    b = W.make_batch(w, seed=7, device=DEV, masked_frac=0.03)
    out = A.awr_loss_fwd_bwd_fused_head(b["hidden"], b["w_head"], b["target_ids"], b["behave_lp"], b["prox_lp"],
                                        b["step_off"], b["traj_off"], b["group_off"], b["rewards"],
                                        want=A.api.HEAD_OPTIONAL_OUTPUTS + ("token_entropy",),
                                        **dict(b["params"], kernel=kernel))
    torch.cuda.synchronize()
    assert int(out["err_word"][0]) == 0
    return float(out["loss"][0])


def main():
    print("config 0 (fp32, generic):", rows_case(W.workload(0), A.KERNEL_GENERIC))
    big = W.workload(3, n_groups=6, group_size=4, n_tok=300)            # V = 151,936 bf16
    for name, k in (("generic", A.KERNEL_GENERIC), ("cluster", A.KERNEL_CLUSTER),
                    ("cluster_rf", A.KERNEL_CLUSTER_RF), ("cluster_rf4", A.KERNEL_CLUSTER_RF4),
                    ("cluster_rfs", A.KERNEL_CLUSTER_RFS), ("cluster_rfs_late", A.KERNEL_CLUSTER_RFS_LATE)):
        print("300 x 151,936 bf16,", name, ":", rows_case(big, k))
    print("300 x 151,936 bf16, cluster_rf + entropy:", rows_case(big, A.KERNEL_CLUSTER_RF, entropy=True))
    for ent in (False, True):
        print("300 x 151,936 bf16, forward stream, entropy", ent, ":",
              rows_case(big, A.KERNEL_FWD_STREAM, backward=False, entropy=ent))
    for name, k in (("1cta recompute", A.KERNEL_HEAD_1CTA), ("2cta recompute", A.KERNEL_HEAD_2CTA),
                    ("2cta stored fp32", A.KERNEL_HEAD_2CTA_STORED), ("2cta E16", A.KERNEL_HEAD_2CTA_E16),
                    ("2cta row reference", A.KERNEL_HEAD_2CTA_ROWREF)):
        print("fused head 600 x 128 x 2056,", name, ":", head_case(k))
    print("SANITIZER_CASES_DONE")


if __name__ == "__main__":
    main()
