"""CPU ORACLE for C4v-symmetric CTMRG (standard eigen-CTMRG and QR-CTMRG).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs may import this package.  It
shares no code with `paper_2505_00494_b200/` (the CUDA path) and never imports
it; only the seeded input generators (`qrctm_inputs`) serve both sides.

Plain NumPy FP64, `reshape` + `@` for every contraction (a library matmul is a
step; no blocking, fusion or reordering beyond what the equations state).  Each
function cites the passage of /root/reference/PAPER.md it follows and the
equation label (E0..E6) of SURVEY.md §8.0, which is the index-form
reconstruction of the paper's Fig. 1 (the figure itself is an unreadable image;
the readings A1..A14 taken are listed in DESIGN.md).

Conventions.  b = D^2.  All arrays C-order.
  a[u,l,d,r]   double-layer site tensor, legs cyclic up/left/down/right, each the
               fused (ket,bra) pair  u = u_ket*D + u_bra.
  C[j,i]       corner, symmetric.        T[i,s,k]  edge, T[i,s,k] = T[k,s,i].
  Q[(j,u),n]   chi*b x chi isometry.     R[n,k]    chi x chi upper triangular.

Parity pins (tests/test_oracle_pins.py): P1 QR structure, P2 Fig.1(f) identity,
P3 symmetry, P4 fn.[47] parameter count, P5/P6 product states, P7 Onsager's
closed form for the 2D Ising partition function, P8 QR vs eigen branch, P9 brute
force finite patches, P10 scale covariance.  `kappa` has no value printed in the
paper; it is pinned by P5-P7, P9.  The paper's energies / timings: parity unpinned
(they need optimised tensors that are not available).
"""
from __future__ import annotations

import numpy as np


# --------------------------------------------------------------------------- E0
def build_a(A: np.ndarray) -> np.ndarray:
    """(E0) a[(u u'),(l l'),(d d'),(r r')] = sum_s A[s,u,l,d,r] A[s,u',l',d',r'].

    PAPER.md:18 ("Contracting each tensor A with its conjugate A^dagger ...
    results in a square lattice network of a tensors"), Fig. 1(b) PAPER.md:24.
    A is real, so the conjugate is A itself.
    """
    d, D = A.shape[0], A.shape[1]
    M = A.reshape(d, D ** 4)
    aa = (M.T @ M).reshape(D, D, D, D, D, D, D, D)          # [u,l,d,r,u',l',d',r']
    aa = aa.transpose(0, 4, 1, 5, 2, 6, 3, 7)               # [u,u',l,l',d,d',r,r']
    b = D * D
    return np.ascontiguousarray(aa.reshape(b, b, b, b))


# ------------------------------------------------------------------- QR (E2, A7)
def householder_qr(X: np.ndarray):
    """Unblocked Householder QR of an m x n matrix (m >= n), thin factors.

    PAPER.md:30 "(unpivoted) QR decomposition".  Textbook algorithm (Golub &
    Van Loan Alg. 5.2.1): for each column k, v = x + sign(x0)*||x|| e1,
    H = I - 2 v v^T / (v^T v); R = H_n ... H_1 X; Q = H_1 ... H_n [I;0].
    Written out here so that the library QR used by `qr_step` is cross-checked
    against an independent implementation (pin P1).  No sign fix here.
    """
    m, n = X.shape
    Rw = np.array(X, dtype=np.float64, copy=True)
    vs = []
    for k in range(n):
        x = Rw[k:, k].copy()
        nrm = np.sqrt(np.sum(x * x))
        v = x.copy()
        if nrm == 0.0:
            vs.append(None)
            continue
        v[0] += nrm if x[0] >= 0.0 else -nrm
        vv = np.sum(v * v)
        Rw[k:, k:] -= np.outer(v, (2.0 / vv) * (v @ Rw[k:, k:]))
        Rw[k + 1:, k] = 0.0
        vs.append((v, vv))
    Q = np.zeros((m, n))
    Q[:n, :n] = np.eye(n)
    for k in range(n - 1, -1, -1):
        if vs[k] is None:
            continue
        v, vv = vs[k]
        Q[k:, :] -= np.outer(v, (2.0 / vv) * (v @ Q[k:, :]))
    return Q, np.triu(Rw[:n, :])


def fix_r_sign(Q: np.ndarray, R: np.ndarray):
    """A7: flip signs so that diag(R) >= 0 (R_kk == 0 counts as +), which makes
    the full-column-rank QR unique.  Q <- Q diag(s), R <- diag(s) R."""
    s = np.where(np.diag(R) < 0.0, -1.0, 1.0)
    return Q * s[None, :], R * s[:, None]


def qr_pos(X: np.ndarray, use_own: bool = False):
    """(E2) c~ = Q R with diag(R) >= 0.  Library QR by default (PAPER.md:30 used a
    library QR), own Householder when `use_own`."""
    if use_own:
        Q, R = householder_qr(X)
    else:
        Q, R = np.linalg.qr(X, mode="reduced")
        R = np.triu(R)
    return fix_r_sign(Q, R)


# ---------------------------------------------------------- growth contractions
def reduced_corner(C: np.ndarray, T: np.ndarray) -> np.ndarray:
    """(E1) X[j,u,k] = sum_i C[j,i] T[i,u,k], returned as the (chi*b) x chi matrix
    c~ with row (j,u) and column k.  PAPER.md:28 ("lower-rank approximation c~ of
    C~ ... reducing the system size in the vertical direction by one row"),
    Fig. 1(e).  Leg grouping: reading A1."""
    chi, b, _ = T.shape
    return (C @ T.reshape(chi, b * chi)).reshape(chi * b, chi)


def half_absorb(Q: np.ndarray, T: np.ndarray) -> np.ndarray:
    """P[u,m,l,J] = sum_j Q[j,u,m] T[j,l,J]   (first factor of (E3)).
    Q is (chi*b) x n with rows (j,u); n may differ from chi (eigen branch)."""
    chi, b, _ = T.shape
    n = Q.shape[1]
    Qm = Q.reshape(chi, b * n)                        # [j,(u,m)]
    P = Qm.T @ T.reshape(chi, b * chi)                # [(u,m),(l,J)]
    return P.reshape(b, n, b, chi)


def absorb_a(P: np.ndarray, a: np.ndarray) -> np.ndarray:
    """S[m,J,d,r] = sum_{u,l} P[u,m,l,J] a[u,l,d,r]   (second factor of (E3))."""
    b, n, _, chi = P.shape
    Pm = P.transpose(1, 3, 0, 2).reshape(n * chi, b * b)    # [(m,J),(u,l)]
    S = Pm @ a.reshape(b * b, b * b)                         # [(m,J),(d,r)]
    return S.reshape(n, chi, b, b)


def project(S: np.ndarray, Q: np.ndarray) -> np.ndarray:
    """T'[m,r,n] = sum_{J,d} S[m,J,d,r] Q[(J,d),n]   (last factor of (E3)).
    PAPER.md:32: "The leading scaling chi^3 D^4 occurs only in the computation
    of T'"."""
    n, chi, b, _ = S.shape
    Sm = S.transpose(0, 3, 1, 2).reshape(n * b, chi * b)     # [(m,r),(J,d)]
    return (Sm @ Q).reshape(n, b, Q.shape[1])


def edge_update(Q: np.ndarray, T: np.ndarray, a: np.ndarray) -> np.ndarray:
    """(E3) T'[m,r,n] = sum Q[(j,u),m] T[j,l,J] a[u,l,d,r] Q[(J,d),n].
    PAPER.md:24 Fig. 1(c),(e)."""
    return project(absorb_a(half_absorb(Q, T), a), Q)


def corner_accelerated(R: np.ndarray, Tp: np.ndarray, Q: np.ndarray) -> np.ndarray:
    """(E4) C'[p,n] = sum_{m,k,r} R[m,k] T'[m,r,p] Q[(k,r),n].
    PAPER.md:32 "the renormalized corner tensor can be efficiently obtained from
    the contraction of T', R, and Q, as shown in the third diagram in Fig. 1(f),
    with a computational cost that scales only as chi^3 D^2"."""
    chi = R.shape[0]
    b = Tp.shape[1]
    W = R @ Q.reshape(chi, b * chi)                          # W[m,(r,n)]
    return Tp.reshape(chi * b, chi).T @ W.reshape(chi * b, chi)


def enlarged_corner(C: np.ndarray, T: np.ndarray, a: np.ndarray) -> np.ndarray:
    """(E5) C~[(J,d),(k,r)] = sum_{j,u,l} X[j,u,k] T[j,l,J] a[u,l,d,r],
    X = C.T (E1).  PAPER.md:20-26, Fig. 1(d): the chi*b x chi*b block that
    standard CTMRG diagonalises."""
    chi, b, _ = T.shape
    X = reduced_corner(C, T)                                 # [(j,u),k]
    Z = half_absorb(X, T)                                    # Z[u,k,l,J]
    Y = absorb_a(Z, a)                                       # Y[k,J,d,r]
    return np.ascontiguousarray(Y.transpose(1, 2, 0, 3).reshape(chi * b, chi * b))


def corner_standard(Q: np.ndarray, Ct: np.ndarray) -> np.ndarray:
    """(E4') C' = Q^T C~ Q, "the standard diagram on the left-hand side" of
    Fig. 1(f)."""
    return Q.T @ (Ct @ Q)


# ------------------------------------------------------------------- the steps
def qr_step(C, T, a, use_own_qr: bool = False, corner: str = "accelerated"):
    """One QR-CTMRG iteration, un-normalised outputs.

    Order (reading A11): c~ from the OLD C,T (E1); Q,R (E2); T' from the old T
    (E3); C' from the new, un-normalised T', R, Q (E4) -- or (E4') through the
    enlarged corner when corner == "enlarged".
    Returns dict with Cn, Tn (un-normalised C', T'), Q, R and X.
    """
    X = reduced_corner(C, T)
    Q, R = qr_pos(X, use_own=use_own_qr)
    Tn = edge_update(Q, T, a)
    if corner == "accelerated":
        Cn = corner_accelerated(R, Tn, Q)
    elif corner == "enlarged":
        Cn = corner_standard(Q, enlarged_corner(C, T, a))
    else:
        raise ValueError(corner)
    return dict(Cn=Cn, Tn=Tn, Q=Q, R=R, X=X)


def eig_step(C, T, a, chi_new: int | None = None):
    """One standard C4v CTMRG iteration (E6), PAPER.md:20-26 and Fig. 1(d):
    diagonalise the enlarged corner C~, keep the chi eigenvectors "with the
    largest magnitudes" (stable sort on -|lambda|, reading A9), C' = U^T C~ U =
    diag(lambda_sel), T' = (E3) with U for Q.  Sign gauge of U: the largest-
    magnitude component of every column is made positive."""
    chi, b, _ = T.shape
    if chi_new is None:
        chi_new = chi
    Ct = enlarged_corner(C, T, a)
    Ct = 0.5 * (Ct + Ct.T)
    lam, V = np.linalg.eigh(Ct)
    sel = np.argsort(-np.abs(lam), kind="stable")[:chi_new]
    U = V[:, sel].copy()
    for c in range(U.shape[1]):
        i = int(np.argmax(np.abs(U[:, c])))
        if U[i, c] < 0.0:
            U[:, c] = -U[:, c]
    Tn = edge_update(U, T, a)
    return dict(Cn=np.diag(lam[sel]), Tn=Tn, U=U, lam=lam[sel])


def normalize(Cn, Tn):
    """Reading A5 (the paper is silent; north_star "then normalizes"): symmetrise
    (an exact no-op in exact arithmetic, pin P3) and divide by the Frobenius
    norm.  C <- (C'+C'^T)/2 / ||.||_F ;  T[i,s,k] <- (T'[i,s,k]+T'[k,s,i])/2 / ||.||_F."""
    C = 0.5 * (Cn + Cn.T)
    T = 0.5 * (Tn + Tn.transpose(2, 1, 0))
    C = C / np.sqrt(np.sum(C * C))
    T = T / np.sqrt(np.sum(T * T))
    return C, T


def spectrum(C):
    """Reading A6: descending singular values of the Frobenius-normalised,
    symmetric corner = sorted |eigenvalues|.  Sum of squares is 1."""
    w = np.linalg.eigvalsh(0.5 * (C + C.T))
    return np.sort(np.abs(w))[::-1]


def run(C0, T0, a, kind: str = "qr", max_iter: int = 100, tol: float = 1e-10,
        use_own_qr: bool = False, corner: str = "accelerated"):
    """Iteration driver ("repeated until convergence is reached";
    criterion = reading A6): C,T start from the normalised C0,T0;
    s_prev = spectrum(C0); each iteration: step, normalize, s = spectrum(C),
    delta = max_i |s_i - s_prev_i|, stop when delta < tol.
    Returns (C, T, iters_done, delta, history_of_delta)."""
    C, T = normalize(C0, T0)
    s_prev = spectrum(C)
    delta = np.inf
    hist = []
    it = 0
    for it in range(1, max_iter + 1):
        if kind == "qr":
            o = qr_step(C, T, a, use_own_qr=use_own_qr, corner=corner)
        elif kind == "eig":
            o = eig_step(C, T, a)
        else:
            raise ValueError(kind)
        C, T = normalize(o["Cn"], o["Tn"])
        s = spectrum(C)
        delta = float(np.max(np.abs(s - s_prev)))
        hist.append(delta)
        s_prev = s
        if delta < tol:
            break
    return C, T, it, delta, hist


# ------------------------------------------------------------ observables (A8)
def kappa_parts(C, T, a):
    """Z4, Z2, Z1 of reading A8: the 2x2 corner network Tr C^4, the 2x3 network
    CTC/CTC and the 3x3 network CTC / TaT / CTC."""
    chi, b, _ = T.shape
    C2 = C @ C
    Z4 = float(np.trace(C2 @ C2))
    E = ((C @ T.reshape(chi, b * chi)).reshape(chi * b, chi) @ C).reshape(chi, b, chi)
    Z2 = float(np.sum(E * E))
    # Z1 = sum E[a,u,c] T[a,l,a'] a[u,l,d,r] T[c,r,c'] E[a',d,c']
    # step 1: F[u,c,l,a'] = sum_a E[a,u,c] T[a,l,a']
    F = (E.reshape(chi, b * chi).T @ T.reshape(chi, b * chi)).reshape(b, chi, b, chi)
    # step 2: G[c,a',d,r] = sum_{u,l} F[u,c,l,a'] a[u,l,d,r]
    G = (F.transpose(1, 3, 0, 2).reshape(chi * chi, b * b) @ a.reshape(b * b, b * b))
    G = G.reshape(chi, chi, b, b)
    # step 3: H[a',d,c'] = sum_{c,r} G[c,a',d,r] T[c,r,c']
    H = (G.transpose(1, 2, 0, 3).reshape(chi * b, chi * b) @ T.reshape(chi * b, chi))
    Z1 = float(np.sum(H.reshape(chi, b, chi) * E))
    return Z4, Z2, Z1


def kappa(C, T, a):
    """Norm per site (reading A8): kappa = Z1 * Z4 / Z2^2.  Site counting:
    (2L+1)^2 + (2L)^2 - 2 (2L+1)(2L) = 1; independent of the scale of C and T."""
    Z4, Z2, Z1 = kappa_parts(C, T, a)
    return Z1 * Z4 / (Z2 * Z2)


# ------------------------------------------------------ paper's initialisation
def bulk_init(A):
    """fn.[48] PAPER.md:132: "we initialize the boundary from the bulk tensors by
    contracting the corresponding bra- and ket- legs on the open boundary".
      C0[(d d'),(r r')]          = sum_{s,u,l} A[s,u,l,d,r] A[s,u,l,d',r']
      T0[(l l'),(d d'),(r r')]   = sum_{s,u}   A[s,u,l,d,r] A[s,u,l',d',r']
    T0's chi legs are (l l') and (r r'), its D^2 leg is (d d')."""
    d, D = A.shape[0], A.shape[1]
    b = D * D
    M = A.reshape(d * D * D, D * D)                     # [(s,u,l),(d,r)]
    C0 = (M.T @ M).reshape(D, D, D, D).transpose(0, 2, 1, 3).reshape(b, b)
    M2 = A.reshape(d * D, D ** 3)                       # [(s,u),(l,d,r)]
    t = (M2.T @ M2).reshape(D, D, D, D, D, D)           # [l,d,r,l',d',r']
    T0 = t.transpose(0, 3, 1, 4, 2, 5).reshape(b, b, b)
    return np.ascontiguousarray(C0), np.ascontiguousarray(T0)


# --------------------------------------- naive loops for tiny sizes (pins only)
def naive_qr_step_tensors(C, T, a, Q, R):
    """(E3) and (E4) as literal index loops -- for tiny chi,b only.  Serves to
    pin the reshape/transposes of edge_update / corner_accelerated."""
    chi, b, _ = T.shape
    Q3 = Q.reshape(chi, b, chi)
    Tn = np.zeros((chi, b, chi))
    for m in range(chi):
        for r in range(b):
            for n in range(chi):
                acc = 0.0
                for j in range(chi):
                    for u in range(b):
                        for l in range(b):
                            for J in range(chi):
                                for dd in range(b):
                                    acc += (Q3[j, u, m] * T[j, l, J] *
                                            a[u, l, dd, r] * Q3[J, dd, n])
                Tn[m, r, n] = acc
    Cn = np.zeros((chi, chi))
    for p in range(chi):
        for n in range(chi):
            acc = 0.0
            for m in range(chi):
                for k in range(chi):
                    for r in range(b):
                        acc += R[m, k] * Tn[m, r, p] * Q3[k, r, n]
            Cn[p, n] = acc
    return Cn, Tn


# ------------------------------------------------- NEXT-3: nearest-neighbour energy
def build_a_pair(A, s, sp):
    """Double-layer tensor with the physical legs left open:
    a^{s s'}[(u u'),(l l'),(d d'),(r r')] = A[s,u,l,d,r] A[s',u',l',d',r']  (sum_s a^{ss} = a of (E0))."""
    D = A.shape[1]
    aa = np.multiply.outer(A[s], A[sp])                       # [u,l,d,r,u',l',d',r']
    aa = aa.transpose(0, 4, 1, 5, 2, 6, 3, 7)
    b = D * D
    return np.ascontiguousarray(aa.reshape(b, b, b, b))


def half_network(C, T, a_x):
    """Left half of the two-site network  C T T C / T a a T / C T T C  cut through the bond between
    the two sites:  LH[k,x,k'] = sum c~[(j,u),k] T[j,l,J] a_x[u,l,d,x] c~[(J,d),k'],  c~ = C.T (E1),
    i.e. (E3) with c~ in place of Q.  k / k' are the top / bottom chi legs, x the cut bond."""
    X = reduced_corner(C, T)
    return edge_update(X, T, a_x)


def rdm2(C, T, A):
    """Two-site reduced density matrix on a nearest-neighbour bond (un-normalised):
    rho[s1,s1',s2,s2'] = sum_{k,x,k'} LH^{s1 s1'}[k,x,k'] LH^{s2 s2'}[k,x,k'].
    The right half is the mirror image of the left one (A is invariant under the l <-> r reflection
    of C4v), so it is the same tensor with the same leg labels."""
    d = A.shape[0]
    LH = [[half_network(C, T, build_a_pair(A, s, sp)) for sp in range(d)] for s in range(d)]
    rho = np.zeros((d, d, d, d))
    for s1 in range(d):
        for s1p in range(d):
            for s2 in range(d):
                for s2p in range(d):
                    rho[s1, s1p, s2, s2p] = np.sum(LH[s1][s1p] * LH[s2][s2p])
    return rho


def energy_nn(C, T, A, H):
    """<h> on one bond for a two-site operator H[(s1 s2),(s1' s2')] (d^2 x d^2, ket index first):
    Tr(rho2 h) / Tr(rho2).  PAPER.md:38-40 evaluates the energy per site of nearest-neighbour
    Hamiltonians this way (the square lattice has two bonds per site; under C4v all bonds are equal)."""
    d = A.shape[0]
    rho = rdm2(C, T, A)
    H4 = np.asarray(H, dtype=np.float64).reshape(d, d, d, d)   # [s1,s2,s1',s2']
    num = np.einsum("abcd,acbd->", rho, H4)                    # rho[s1,s1',s2,s2'] H[s1,s2,s1',s2']
    den = np.einsum("aabb->", rho)
    return float(num / den)
