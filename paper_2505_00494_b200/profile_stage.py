"""Run a few QR-CTMRG steps of one config so that a profiler can pick a stage by
its NVTX range (K1_reduced_corner ... K7_normalize), e.g.

  ncu --set full --nvtx --nvtx-include "K4_absorb_a/" -c 1 \
      python -m paper_2505_00494_b200.profile_stage --config cfg4 --steps 2

--warmup N runs the NEXT-2 warm-up instead (bulk initialisation + N eigen steps, NVTX ranges
E1_enlarged_corner, E2_eigh, E3_edge); --eig-steps M adds M eigen steps at the final chi.
"""
import argparse
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def main():
    import torch
    import paper_2505_00494_b200 as pkg
    from qrctm_inputs import CONFIGS, gen_named
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="cfg4", choices=sorted(CONFIGS))
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=-1)
    ap.add_argument("--eig-steps", type=int, default=0)
    ap.add_argument("--qr-path", type=int, default=0, help="QRCTM_OPT_QR_PATH (0 automatic / CholeskyQR2, 2 blocked Householder, ...)")
    ap.add_argument("--absorb-mode", type=int, default=0, help="QRCTM_OPT_ABSORB_MODE")
    a = ap.parse_args()
    A, C0, T0, c = gen_named(a.config)
    h = pkg.QRCTM(c["d"], c["D"], c["chi"])
    h.set_option(pkg.OPT_USE_GRAPH, 0)          # plain launches keep the NVTX stage ranges
    h.set_option(pkg.OPT_QR_PATH, a.qr_path)
    h.set_option(pkg.OPT_ABSORB_MODE, a.absorb_mode)
    h.set_A(A)
    if a.warmup >= 0:
        h.warmup(a.warmup)
    else:
        h.set_env(C0, T0)
    for _ in range(a.eig_steps):
        h.eig_step()
    for _ in range(a.steps):
        h.step()
    torch.cuda.synchronize()
    print(a.config, "steps", a.steps, "launches", h.launch_count(), "spectrum[0:3]", h.get_corner_spectrum()[:3])
    h.close()


if __name__ == "__main__":
    main()
