"""Demo: free energy per site of the square-lattice Ising model with QR-CTMRG on the GPU.

The partition function is the norm of a d = 2, D = 2 C4v-symmetric iPEPS ("QR-CTMRG can also be
applied to contract 2D tensor networks in the context of classical 2D partition functions"):
A[s,u,l,d,r] = w_su w_sl w_sd w_sr with w = sqrt(B), B = [[e^{K/2}, e^{-K/2}], [e^{-K/2}, e^{K/2}]], so that
kappa = norm per site = Z^(1/N).  Compared with Onsager's closed form.

    python -m paper_2505_00494_b200.demo_ising --K 0.3 --chi 16
"""
import argparse
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def ising_tensor(K):
    B = np.array([[np.exp(K / 2), np.exp(-K / 2)], [np.exp(-K / 2), np.exp(K / 2)]])
    lam, V = np.linalg.eigh(B)
    w = (V * np.sqrt(lam)) @ V.T
    return np.ascontiguousarray(np.einsum("su,sl,sd,sr->suldr", w, w, w, w))


def onsager(K, n=2048):
    t = (np.arange(n) + 0.5) * (2 * np.pi / n)
    c = np.cos(t)
    f = np.log(np.cosh(2 * K) ** 2 - np.sinh(2 * K) * (c[:, None] + c[None, :]))
    return float(np.log(2.0) + 0.5 * f.mean())


def main():
    import paper_2505_00494_b200 as pkg
    from qrctm_inputs import gen_config
    ap = argparse.ArgumentParser()
    ap.add_argument("--K", type=float, default=0.3)
    ap.add_argument("--chi", type=int, default=16)
    ap.add_argument("--max-iter", type=int, default=400)
    a = ap.parse_args()
    _, C0, T0 = gen_config(2, 2, a.chi, 1)            # random symmetric start
    h = pkg.QRCTM(2, 2, a.chi)
    h.set_A(ising_tensor(a.K))
    h.set_env(C0, T0)
    it, delta = h.run(a.max_iter, 1e-13)
    lnk = float(np.log(h.norm_per_site()))
    print(f"K = {a.K}, chi = {a.chi}: {it} QR-CTMRG iterations (delta {delta:.1e}), ln kappa = {lnk:.13f}, "
          f"Onsager {onsager(a.K):.13f}, difference {lnk - onsager(a.K):+.1e}")
    h.close()


if __name__ == "__main__":
    main()
