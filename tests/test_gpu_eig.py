"""GPU parity for NEXT-2: the paper's boundary initialisation from the
bulk tensor (fn.[48] PAPER.md:132), the standard eigen step with the library's
own top-k symmetric eigensolver, and the warm-up with chi growth.

Eigenvectors are only defined up to eps * ||A|| / gap: two correct eigensolvers (LAPACK inside the
oracle, csrc/eigh.cuh on the GPU) differ by that much, so tolerances on U and T' are derived from
the measured gaps of each case; eigenvalues, orthonormality and residuals are held to rounding."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import paper_2505_00494_b200 as pkg
from oracle import ctmrg as o
from qrctm_inputs import gen_config

EPS = np.finfo(np.float64).eps


def rel(x, y):
    x = np.asarray(x); y = np.asarray(y)
    return np.linalg.norm(x - y) / np.linalg.norm(y)


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2505_00494_b200 import build as b
    b.build()


def torch_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def lapack_top(A, k):
    """the oracle's selection and gauge (oracle/ctmrg.py eig_step) on a plain symmetric matrix"""
    lam, V = np.linalg.eigh(A)
    sel = np.argsort(-np.abs(lam), kind="stable")[:k]
    U = V[:, sel].copy()
    for c in range(k):
        i = int(np.argmax(np.abs(U[:, c])))
        if U[i, c] < 0:
            U[:, c] = -U[:, c]
    # smallest distance from a selected eigenvalue to any other eigenvalue
    gaps = np.diff(lam)
    gl = np.concatenate(([np.inf], gaps)); gr = np.concatenate((gaps, [np.inf]))
    gap = np.minimum(gl, gr)[sel]
    return lam[sel], U, gap


def check_eigh(A, k, lam, U):
    n = A.shape[0]
    nrm = np.linalg.norm(A, 2)
    lo, Uo, gap = lapack_top(A, k)
    assert np.max(np.abs(lam - lo)) < 8 * n * EPS * nrm
    assert np.linalg.norm(U.T @ U - np.eye(k)) < 50 * k * EPS
    assert np.linalg.norm(A @ U - U * lam) < 30 * n * EPS * nrm * np.sqrt(k)
    for c in range(k):
        assert U[np.argmax(np.abs(U[:, c])), c] > 0
        tol = 100 * EPS * nrm / gap[c]
        if tol < 1e-3:       # direction defined well enough to compare with LAPACK's
            assert np.linalg.norm(U[:, c] - Uo[:, c]) < max(tol, 1e-13), (c, gap[c])


@pytest.mark.parametrize("n,k", [(1, 1), (2, 1), (2, 2), (3, 2), (5, 5), (16, 8), (81, 36), (256, 64), (300, 300),
                                 (625, 100), (1037, 33), (2401, 196)])
def test_eigh_top_matches_lapack(n, k):
    g = np.random.default_rng(n * 31 + k)
    A = g.standard_normal((n, n)); A = 0.5 * (A + A.T)
    lam, U = pkg.eigh_top_f64(torch_dev(A), k)
    check_eigh(A, k, lam.cpu().numpy(), U.cpu().numpy())


def test_eigh_top_decaying_spectrum_and_sign_pairs():
    """a corner-like spectrum: geometric decay over 12 decades with +/- pairs (hazard H2)"""
    g = np.random.default_rng(5)
    n, k = 200, 40
    Qm, _ = np.linalg.qr(g.standard_normal((n, n)))
    lam = np.array([(-1) ** i * 10.0 ** (-12.0 * (i // 2) / (n // 2)) * (1 + 0.01 * (i % 2)) for i in range(n)])
    A = (Qm * lam) @ Qm.T; A = 0.5 * (A + A.T)
    l, U = pkg.eigh_top_f64(torch_dev(A), k)
    check_eigh(A, k, l.cpu().numpy(), U.cpu().numpy())


def test_eigh_top_degenerate_multiplets():
    """exactly repeated eigenvalues (symmetry multiplets): any orthonormal basis of the eigenspace is
    correct -- compare the eigenspace projectors, orthonormality and residual"""
    g = np.random.default_rng(11)
    n = 120
    Qm, _ = np.linalg.qr(g.standard_normal((n, n)))
    vals = np.concatenate(([5.0] * 3, [-4.0] * 2, [3.0], [2.5] * 4, 0.1 * g.standard_normal(n - 10)))
    A = (Qm * vals) @ Qm.T; A = 0.5 * (A + A.T)
    k = 10
    l, U = pkg.eigh_top_f64(torch_dev(A), k)
    l, U = l.cpu().numpy(), U.cpu().numpy()
    assert np.max(np.abs(l - vals[:k])) < 1e-12
    assert np.linalg.norm(U.T @ U - np.eye(k)) < 1e-12
    assert np.linalg.norm(A @ U - U * l) < 1e-11
    for lo_, hi_ in [(0, 3), (3, 5), (5, 6), (6, 10)]:
        P = U[:, lo_:hi_] @ U[:, lo_:hi_].T
        Po = Qm[:, lo_:hi_] @ Qm[:, lo_:hi_].T
        assert np.linalg.norm(P - Po) < 1e-10


def test_eigh_top_already_tridiagonal_and_diagonal():
    """tau = 0 reflectors (nothing to eliminate) and a reducible tridiagonal (zero off-diagonals)"""
    g = np.random.default_rng(2)
    n = 40
    D = np.diag(g.standard_normal(n))
    l, U = pkg.eigh_top_f64(torch_dev(D), 7)
    check_eigh(D, 7, l.cpu().numpy(), U.cpu().numpy())
    Tm = np.diag(g.standard_normal(n)) + np.diag(g.standard_normal(n - 1), 1)
    Tm = np.triu(Tm) + np.triu(Tm, 1).T
    l, U = pkg.eigh_top_f64(torch_dev(Tm), 11)
    check_eigh(Tm, 11, l.cpu().numpy(), U.cpu().numpy())


def test_eigh_rejects_bad_sizes():
    lib = pkg.load_library()
    assert lib.qrctm_eigh_work_bytes(0, 1) == 0 and lib.qrctm_eigh_work_bytes(5, 6) == 0
    assert lib.qrctm_eigh_work_bytes(14001, 10) == 0 and lib.qrctm_eigh_work_bytes(100, 10) > 0


# ------------------------------------------------------------------ bulk initialisation, eigen step
@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (2, 3, 36, 1), (3, 2, 4, 7), (2, 4, 16, 2), (2, 1, 1, 3)])
def test_bulk_init_matches_oracle(d, D, chi, seed):
    A, _, _ = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A)
    h.init_bulk()
    assert h.chi == D * D and h.chi_cap == chi
    C, T = h.get_env()
    Co, To = o.normalize(*o.bulk_init(A))
    assert C.shape == Co.shape and T.shape == To.shape
    assert rel(C, Co) < 1e-13 and rel(T, To) < 1e-13
    h.close()


def test_bulk_init_needs_room():
    A, _, _ = gen_config(2, 3, 5, 0)
    h = pkg.QRCTM(2, 3, 5)
    h.set_A(A)
    with pytest.raises(pkg.QrctmError):
        h.init_bulk()           # D^2 = 9 > chi = 5
    h.close()


def _align(U, Uo):
    """Column signs s with U * s ~ Uo.  The oracle's gauge (largest-|.| component positive) is decided by
    rounding when two components tie -- e.g. the bulk-initialised C~ commutes with the ket<->bra swap, so its
    antisymmetric eigenvectors have +x / -x pairs -- hence C', T' are compared modulo this sign gauge
    (U -> U s, T' -> s T' s, C' = diag(lambda) unchanged), which every later step is covariant under."""
    s = np.sign(np.sum(U * Uo, axis=0))
    s[s == 0] = 1.0
    return s


def _gauge(C, T, s):
    return C * s[:, None] * s[None, :], T * s[:, None, None] * s[None, None, :]


def _eig_tol(Ct, chi_new):
    """eps * ||C~|| / (smallest gap around a kept eigenvalue), with slack for the two contractions"""
    lam = np.linalg.eigvalsh(0.5 * (Ct + Ct.T))
    sel = np.argsort(-np.abs(lam), kind="stable")[:chi_new]
    gaps = np.diff(lam)
    gl = np.concatenate(([np.inf], gaps)); gr = np.concatenate((gaps, [np.inf]))
    gap = np.minimum(gl, gr)[sel].min()
    return max(1e-11, 100 * EPS * np.abs(lam).max() / gap)


@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (2, 3, 36, 1), (3, 2, 6, 7), (2, 4, 64, 2), (2, 3, 7, 8)])
def test_eig_step_matches_oracle(d, D, chi, seed):
    """same chi in and out, from the seeded random environment"""
    A, C0, T0 = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0)
    h.eig_step()
    U, lam = h.get_eig()
    Cn, Tn = h.get_raw()
    C, T = h.get_env()
    h.close()
    a = o.build_a(A)
    Cr, Tr = o.normalize(C0, T0)
    s = o.eig_step(Cr, Tr, a)
    tol = _eig_tol(o.enlarged_corner(Cr, Tr, a), chi)
    assert tol < 1e-6
    assert np.max(np.abs(lam - s["lam"])) < 1e-13 * np.abs(s["lam"]).max() * chi * D * D
    assert np.linalg.norm(U.T @ U - np.eye(chi)) < 50 * chi * EPS
    sg = _align(U, s["U"])
    assert rel(U * sg, s["U"]) < tol
    Cn, Tn = _gauge(Cn, Tn, sg); C, T = _gauge(C, T, sg)
    assert rel(Cn, s["Cn"]) < 1e-12 and rel(Tn, s["Tn"]) < tol
    Co, To = o.normalize(s["Cn"], s["Tn"])
    assert rel(C, Co) < 1e-12 and rel(T, To) < tol


@pytest.mark.parametrize("d,D,chi,seed", [(2, 2, 8, 0), (2, 2, 16, 1), (2, 3, 36, 1), (2, 3, 81, 4), (3, 2, 13, 7),
                                          (2, 4, 64, 2)])
def test_warmup_growth_matches_oracle(d, D, chi, seed):
    """bulk initialisation, then one eigen step growing chi from D^2 to min(chi, D^4)"""
    A, _, _ = gen_config(d, D, chi, seed)
    b = D * D
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A)
    h.warmup(1)
    chi1 = min(chi, b * b)
    assert h.chi == chi1
    U, lam = h.get_eig()
    C, T = h.get_env()
    a = o.build_a(A)
    Cr, Tr = o.normalize(*o.bulk_init(A))
    s = o.eig_step(Cr, Tr, a, chi_new=chi1)
    tol = _eig_tol(o.enlarged_corner(Cr, Tr, a), chi1)
    assert tol < 1e-5
    assert U.shape == s["U"].shape == (b * b, chi1)
    assert np.max(np.abs(lam - s["lam"])) < 1e-13 * np.abs(s["lam"]).max() * b * b
    sg = _align(U, s["U"])
    assert rel(U * sg, s["U"]) < tol
    Co, To = o.normalize(s["Cn"], s["Tn"])
    assert C.shape == Co.shape and T.shape == To.shape
    C, T = _gauge(C, T, sg)
    assert rel(C, Co) < 1e-12 and rel(T, To) < tol
    # a QR step at the grown chi continues from there (the handle's shapes follow the current chi)
    if chi1 == chi:
        h.step()
        C2, T2 = _gauge(*h.get_env(), sg)
        q = o.qr_step(Co, To, a)
        C2o, T2o = o.normalize(q["Cn"], q["Tn"])
        cond = np.linalg.cond(q["X"])
        assert rel(C2, C2o) < tol * max(cond, 10) and rel(T2, T2o) < tol * max(cond, 10)
    h.close()


def test_warmup_then_qr_run_converges_to_the_same_fixed_point():
    """eigen warm-up, then QR-CTMRG; the converged norm per site does not depend on how the
    environment was initialised (random start vs bulk start)"""
    d, D, chi, seed = 2, 2, 16, 5
    A, C0, T0 = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A)
    h.warmup(2)
    assert h.chi == chi
    it, dl = h.run(400, 1e-12)
    k1 = h.norm_per_site()
    s1 = h.get_corner_spectrum()
    h.set_env(C0, T0)
    it2, dl2 = h.run(400, 1e-12)
    k2 = h.norm_per_site()
    h.close()
    a = o.build_a(A)
    Cr, Tr = o.normalize(*o.bulk_init(A))
    for chi_new in (16, 16):
        s = o.eig_step(Cr, Tr, a, chi_new=min(chi_new, Cr.shape[0] * D * D))
        Cr, Tr = o.normalize(s["Cn"], s["Tn"])
    Co, To, ito, dlo, _ = o.run(Cr, Tr, a, kind="qr", max_iter=400, tol=1e-12)
    ko = o.kappa(Co, To, a)
    assert dl < 1e-10 and dlo < 1e-10
    assert abs(k1 / ko - 1) < 1e-9
    so = o.spectrum(Co)
    assert np.max(np.abs(s1[:10] - so[:10]) / so[:10]) < 1e-8
    if dl2 < 1e-10:
        assert abs(k1 / k2 - 1) < 1e-6


def test_eig_step_argument_errors():
    A, C0, T0 = gen_config(2, 2, 8, 0)
    h = pkg.QRCTM(2, 2, 8)
    with pytest.raises(pkg.QrctmError):
        h.eig_step()                       # nothing set
    h.set_A(A); h.set_env(C0, T0)
    with pytest.raises(pkg.QrctmError):
        h.eig_step(9)                      # above capacity
    with pytest.raises(pkg.QrctmError):
        h.get_eig()                        # no eigen step yet
    h.eig_step(5)                          # shrinking is allowed
    assert h.chi == 5
    C, T = h.get_env()
    assert C.shape == (5, 5) and T.shape == (5, 4, 5)
    h.set_env(C0, T0)                      # back to capacity
    assert h.chi == 8
    h.close()


def test_observables_follow_the_current_chi():
    """norm per site, corner spectrum and the bond energy right after the bulk initialisation (chi = D^2 < capacity)
    and after the warm-up step, against the oracle on the same environments"""
    d, D, chi, seed = 2, 2, 12, 6
    A, _, _ = gen_config(d, D, chi, seed)
    g = np.random.default_rng(3)
    H = g.standard_normal((d * d, d * d)); H = H + H.T
    a = o.build_a(A)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A)
    h.init_bulk()
    Co, To = o.normalize(*o.bulk_init(A))
    assert abs(h.norm_per_site() / o.kappa(Co, To, a) - 1) < 1e-11
    assert abs(h.energy_nn(H) - o.energy_nn(Co, To, A, H)) < 1e-11
    it, dl = h.run(3, -1.0)                       # QR steps at chi = D^2
    assert it == 3 and h.chi == D * D
    C, T = Co, To
    for _ in range(3):
        q = o.qr_step(C, T, a)
        C, T = o.normalize(q["Cn"], q["Tn"])
    Cg, Tg = h.get_env()
    cond = np.linalg.cond(o.reduced_corner(C, T))
    assert rel(Cg, C) < 1e-12 * max(cond, 10) and rel(Tg, T) < 1e-12 * max(cond, 10)
    assert np.max(np.abs(h.get_corner_spectrum() - o.spectrum(C))) < 1e-11
    h.close()


def test_ising_onsager_through_the_papers_flow():
    """PAPER.md:28 + fn.[48]: bulk initialisation, two eigen steps growing chi 4 -> 16, then QR-CTMRG to convergence;
    ln(kappa) of the Ising partition function against Onsager's closed form (structured A: the enlarged corner is
    rank-deficient, so the kept eigenvectors of the zero cluster are arbitrary -- kappa is gauge-invariant)."""
    from tests.brute import ising_A, onsager_ln_kappa
    K = 0.3
    h = pkg.QRCTM(2, 2, 16)
    h.set_A(ising_A(K))
    h.warmup(2)
    assert h.chi == 16
    it, dl = h.run(300, 1e-13)
    assert abs(np.log(h.norm_per_site()) - onsager_ln_kappa(K)) < 1e-10
    h.close()


def test_eigen_branch_and_qr_branch_agree_at_convergence():
    """PAPER.md:8 "without loss of accuracy": iterating the standard step and iterating the QR step from the same
    start reach the same norm per site and corner spectrum (the GPU's own eigen branch, not the oracle's)."""
    d, D, chi, seed = 2, 2, 8, 0
    A, C0, T0 = gen_config(d, D, chi, seed)
    h = pkg.QRCTM(d, D, chi)
    h.set_A(A); h.set_env(C0, T0)
    it, dl = h.run(500, 1e-12)
    kq, sq = h.norm_per_site(), h.get_corner_spectrum()
    h.set_env(C0, T0)
    s_prev = None
    for n_e in range(200):
        h.eig_step()
        s = np.sort(np.abs(np.diag(h.get_env()[0])))[::-1]        # C' = diag(lambda) / ||.||
        if s_prev is not None and np.max(np.abs(s - s_prev)) < 1e-12:
            break
        s_prev = s
    ke = h.norm_per_site()
    h.close()
    assert dl < 1e-12 and n_e < 199 and n_e < it
    assert abs(kq / ke - 1) < 1e-10
    assert np.max(np.abs(sq - s)) < 1e-9
