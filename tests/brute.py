"""Brute-force helpers for the oracle pins: exact row-by-row contraction of a
finite open-boundary patch of double-layer tensors (fn.[48] PAPER.md:132 closes
the open legs by contracting bra with ket), and Onsager's closed form.
Independent of oracle/ (uses only numpy / scipy.integrate)."""
import numpy as np


def patch_norm(a: np.ndarray, nrows: int, ncols: int, D: int) -> float:
    """<psi|psi> of an nrows x ncols open patch of `a[u,l,d,r]` tensors whose
    outer legs are closed with delta(ket,bra)."""
    b = D * D
    v = np.eye(D).reshape(b)
    state = v
    for _ in range(ncols - 1):
        state = np.multiply.outer(state, v)
    state = state.reshape((b,) * ncols)
    for _ in range(nrows):
        # cur[h, legs...]: horizontal leg first
        cur = np.multiply.outer(v, state)
        for c in range(ncols):
            # contract cur's leg 0 (l) and leg 1+c (u) with a[u,l,d,r]
            cur = np.tensordot(cur, a, axes=([1 + c, 0], [0, 1]))  # legs..., d, r
            # move d to position c and r to the front
            nd = cur.ndim
            order = [nd - 1] + list(range(0, c)) + [nd - 2] + list(range(c, nd - 2))
            cur = cur.transpose(order)
        state = np.tensordot(v, cur, axes=([0], [0]))
    for _ in range(ncols):
        state = np.tensordot(state, v, axes=([0], [0]))
    return float(state)


def onsager_ln_kappa(K: float) -> float:
    """ln of the partition function per site of the square-lattice Ising model at
    coupling K (Onsager 1944):
    ln 2 + 1/(8 pi^2) int int ln[cosh^2 2K - sinh 2K (cos t1 + cos t2)]."""
    n = 2048
    t = (np.arange(n) + 0.5) * (2 * np.pi / n)
    c = np.cos(t)
    f = np.log(np.cosh(2 * K) ** 2 - np.sinh(2 * K) * (c[:, None] + c[None, :]))
    return float(np.log(2.0) + 0.5 * f.mean())


def ising_A(K: float) -> np.ndarray:
    """d=2, D=2 C4v tensor whose norm network is the Ising partition function:
    A[s,u,l,d,r] = w_su w_sl w_sd w_sr, w = sqrt(B) (symmetric matrix square
    root), B = [[e^{K/2}, e^{-K/2}], [e^{-K/2}, e^{K/2}]] so that each lattice
    bond carries (w w^T)_{st}^2 = e^{+-K}."""
    B = np.array([[np.exp(K / 2), np.exp(-K / 2)], [np.exp(-K / 2), np.exp(K / 2)]])
    lam, V = np.linalg.eigh(B)
    w = (V * np.sqrt(lam)) @ V.T
    return np.einsum("su,sl,sd,sr->suldr", w, w, w, w)


def patch_contract(site, nrows: int, ncols: int, D: int) -> float:
    """Like patch_norm but with a possibly different double-layer tensor per site: site(r, c) -> a[u,l,d,r]."""
    b = D * D
    v = np.eye(D).reshape(b)
    state = v
    for _ in range(ncols - 1):
        state = np.multiply.outer(state, v)
    state = state.reshape((b,) * ncols)
    for rr in range(nrows):
        cur = np.multiply.outer(v, state)
        for c in range(ncols):
            cur = np.tensordot(cur, site(rr, c), axes=([1 + c, 0], [0, 1]))
            nd = cur.ndim
            order = [nd - 1] + list(range(0, c)) + [nd - 2] + list(range(c, nd - 2))
            cur = cur.transpose(order)
        state = np.tensordot(v, cur, axes=([0], [0]))
    for _ in range(ncols):
        state = np.tensordot(state, v, axes=([0], [0]))
    return float(state)


def patch_energy_nn(A: np.ndarray, H: np.ndarray, nrows: int, ncols: int, r0: int, c0: int) -> float:
    """<psi|h|psi>/<psi|psi> for an open nrows x ncols patch of the single-site iPEPS tensor A with the
    two-site operator H[(s1 s2),(s1' s2')] on the horizontal bond (r0,c0)-(r0,c0+1).  Brute force."""
    d, D = A.shape[0], A.shape[1]
    b = D * D

    def pair(s, sp):
        aa = np.multiply.outer(A[s], A[sp]).transpose(0, 4, 1, 5, 2, 6, 3, 7)
        return aa.reshape(b, b, b, b)

    a = sum(pair(s, s) for s in range(d))
    H4 = np.asarray(H).reshape(d, d, d, d)
    num = 0.0
    for s1 in range(d):
        for s1p in range(d):
            for s2 in range(d):
                for s2p in range(d):
                    hv = H4[s1, s2, s1p, s2p]
                    if hv == 0.0:
                        continue
                    t1, t2 = pair(s1, s1p), pair(s2, s2p)
                    num += hv * patch_contract(
                        lambda r, c: t1 if (r, c) == (r0, c0) else (t2 if (r, c) == (r0, c0 + 1) else a),
                        nrows, ncols, D)
    return num / patch_contract(lambda r, c: a, nrows, ncols, D)
