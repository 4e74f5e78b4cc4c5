"""Time per CTMRG step against chi at fixed D on the GPU -- the kind of measurement the paper's Fig. 2(b,c) shows
(optimised D = 6 Heisenberg tensor, chi up to 600, QR-CTMRG vs standard CTMRG; the figure itself is
unreadable in the reference, so there is no number to compare with).  Synthetic inputs: the BASELINE.json recipe
(`qrctm_inputs.gen_config`) at the requested D and chi.

Per chi: device time of one QR-CTMRG step (explicit double-layer tensor, and the layered absorption), and -- while the
enlarged corner fits the library's eigensolver (chi D^2 <= 14000) -- of one standard (eigen) step at the same chi.

    python -m paper_2505_00494_b200.chi_sweep --D 6 --chis 100,200,300,400,500,600
"""
import argparse
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def time_steps(h, n, torch):
    """Mean device time (ms) of n QR-CTMRG steps through qrctm_run (graph replay, check every step)."""
    h.run(2, -1.0)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(h.stream)
    h.run(n, -1.0)
    e1.record(h.stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def main():
    import torch
    import paper_2505_00494_b200 as pkg
    from qrctm_inputs import gen_config
    ap = argparse.ArgumentParser()
    ap.add_argument("--d", type=int, default=2)
    ap.add_argument("--D", type=int, default=6)
    ap.add_argument("--chis", default="100,200,300,400,500,600")
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--seed", type=int, default=6)
    ap.add_argument("--eig-max-n", type=int, default=14000)
    a = ap.parse_args()
    b = a.D * a.D
    rows = []
    for chi in [int(x) for x in a.chis.split(",")]:
        A, C0, T0 = gen_config(a.d, a.D, chi, a.seed)
        h = pkg.QRCTM(a.d, a.D, chi)
        h.set_A(A)
        h.set_env(C0, T0)
        row = {"D": a.D, "chi": chi, "m": chi * b}
        row["qr_step_ms"] = time_steps(h, a.steps, torch)
        flops = 2 * chi**3 * b + 4 * chi * b * chi**2 - 4 * chi**3 / 3 + 4 * (chi * b) ** 2 * chi \
            + 2 * chi**2 * b**4 + 4 * chi**3 * b
        row["qr_step_tflops"] = flops / (row["qr_step_ms"] * 1e-3) / 1e12
        if chi % 2 == 0:
            h.set_option(pkg.OPT_ABSORB_MODE, 1)
            h.set_env(C0, T0)
            row["qr_step_layered_ms"] = time_steps(h, a.steps, torch)
            h.set_option(pkg.OPT_ABSORB_MODE, 0)
        if chi * b <= a.eig_max_n:
            h.set_env(C0, T0)
            h.run(2, -1.0)
            h.eig_step()                       # first call allocates the eigensolver workspace
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(h.stream)
            h.eig_step()
            e1.record(h.stream)
            torch.cuda.synchronize()
            row["eig_step_ms"] = e0.elapsed_time(e1)
            row["eig_over_qr"] = row["eig_step_ms"] / row["qr_step_ms"]
        h.close()
        del h
        torch.cuda.empty_cache()
        rows.append(row)
        print(json.dumps(row), flush=True)


if __name__ == "__main__":
    main()
