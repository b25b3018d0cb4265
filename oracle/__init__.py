"""CPU oracle for the LO-AFQMC local energy -- TEST INFRASTRUCTURE, NOT PRODUCT.

Thin ctypes wrapper around oracle/lo_oracle.cpp (plain fp64 loops written from the paper) plus the
glue that strings its steps together.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It shares nothing with the CUDA path
(paper_2202_00832_b200) and never imports it.  Pins: tests/test_oracle_*.py; beyond them the
energies are "parity unpinned" to any number printed by the paper (it prints none).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lo_oracle.cpp")
_LIB = os.path.join(_HERE, "liblo_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/lo_oracle.cpp with g++ (OpenMP) into oracle/liblo_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _l():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def num_threads() -> int:
    return int(_l().orc_num_threads())


# ------------------------------------------------------------------ single steps
def theta(psi, phi):
    """Eq. 15: Theta = Phi (Psi^T Phi)^-1.  Returns (theta [N,O], det(Psi^T Phi), status)."""
    psi, phi = _f64(psi), _c128(phi)
    N, O = psi.shape
    th = np.empty((N, O), dtype=np.complex128)
    det = np.zeros(1, dtype=np.complex128)
    st = _l().orc_theta(C.c_int(N), C.c_int(O), _p(psi), _p(phi), _p(th), _p(det))
    return th, det[0], int(st)


def green(psi, th):
    """Eq. 14: G[p,q] = sum_i Theta[q,i] Psi[p,i]."""
    psi, th = _f64(psi), _c128(th)
    N, O = psi.shape
    G = np.empty((N, N), dtype=np.complex128)
    _l().orc_green(C.c_int(N), C.c_int(O), _p(psi), _p(th), _p(G))
    return G


def energy_bruteforce(h, L, Ga, Gb=None):
    """O1: (E1, E_J, E_K) from Eq. 8 + Eq. 10 with explicit spin sums; closed shell when Gb is None."""
    h, L, Ga = _f64(h), _f64(L), _c128(Ga)
    Gb = Ga if Gb is None else _c128(Gb)
    out = np.zeros(3, dtype=np.complex128)
    _l().orc_energy_bruteforce(C.c_int(h.shape[0]), C.c_int(L.shape[0]), _p(h), _p(L), _p(Ga), _p(Gb), _p(out))
    return out


def half_rotate(L, h, psi):
    """Lbar[g,i,p] = sum_q L[g,p,q] psi[q,i]; hbar[i,p] = sum_q psi[q,i] h[q,p]."""
    L, h, psi = _f64(L), _f64(h), _f64(psi)
    X, N, _ = L.shape
    O = psi.shape[1]
    Lbar = np.empty((X, O, N))
    hbar = np.empty((O, N))
    _l().orc_half_rotate(C.c_int(N), C.c_int(X), C.c_int(O), _p(L), _p(h), _p(psi), _p(Lbar), _p(hbar))
    return Lbar, hbar


def _ptr_array(arrs):
    return (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])


def onebody_coulomb(Lbars, hbars, thetas, want_X=False):
    """(E1, E_J) by the Cholesky route for 1 (closed shell) or 2 (unrestricted) spins; optionally X^g."""
    Lbars = [_f64(a) for a in Lbars]
    hbars = [_f64(a) for a in hbars]
    thetas = [_c128(a) for a in thetas]
    ns = len(Lbars)
    X, _, N = Lbars[0].shape
    O = (C.c_int * ns)(*[a.shape[1] for a in Lbars])
    out = np.zeros(2, dtype=np.complex128)
    Xg = np.zeros(X, dtype=np.complex128)
    _l().orc_onebody_coulomb(C.c_int(N), C.c_int(X), C.c_int(ns), O, _ptr_array(Lbars), _ptr_array(hbars),
                             _ptr_array(thetas), _p(out), _p(Xg))
    return (out[0], out[1], Xg) if want_X else (out[0], out[1])


def propagator(L, x):
    """B[p,q] = sum_g x[g] L[g,p,q] (the propagation matrix of one walker)."""
    L, x = _f64(L), _c128(x)
    X, N, _ = L.shape
    B = np.zeros((N, N), dtype=np.complex128)
    _l().orc_propagator(C.c_int(N), C.c_int(X), _p(L), _p(x), _p(B))
    return B


def exchange_cholesky(Lbar, th):
    """O2 single-spin exchange sum, Eq. 16."""
    Lbar, th = _f64(Lbar), _c128(th)
    X, O, N = Lbar.shape
    out = np.zeros(1, dtype=np.complex128)
    _l().orc_exchange_cholesky(C.c_int(N), C.c_int(X), C.c_int(O), _p(Lbar), _p(th), _p(out))
    return out[0]


def pair_eri(Lbar, i, j):
    """Y^{ij}[p,q] = sum_g Lbar[g,i,p] Lbar[g,j,q]."""
    Lbar = _f64(Lbar)
    X, O, N = Lbar.shape
    Y = np.empty((N, N))
    _l().orc_pair_eri(C.c_int(N), C.c_int(X), C.c_int(O), _p(Lbar), C.c_int(i), C.c_int(j), _p(Y))
    return Y


def exchange_full_eri(Lbar, th):
    """O3 single-spin exchange sum from on-the-fly pair ERI blocks, Eq. 17."""
    Lbar, th = _f64(Lbar), _c128(th)
    X, O, N = Lbar.shape
    out = np.zeros(1, dtype=np.complex128)
    _l().orc_exchange_full_eri(C.c_int(N), C.c_int(X), C.c_int(O), _p(Lbar), _p(th), _p(out))
    return out[0]


def svd(A):
    """One-sided Jacobi SVD.  Returns (Ut [n,n] rows = left vectors, s descending, Wt [n,n] rows = right vectors)."""
    A = _f64(A)
    n = A.shape[0]
    Ut, s, Wt = np.empty((n, n)), np.empty(n), np.empty((n, n))
    _l().orc_svd(C.c_int(n), _p(A), _p(Ut), _p(s), _p(Wt))
    return Ut, s, Wt


# ------------------------------------------------------------------ factor sets
@dataclass
class FactorSet:
    """Truncated factors of one spin: pairs (pi[k] <= pj[k]) with rank r[k]; rows of pair k start at off[k]."""
    N: int
    O: int
    pi: np.ndarray
    pj: np.ndarray
    r: np.ndarray
    off: np.ndarray
    U: np.ndarray        # [sum r, N]
    sigma: np.ndarray    # [sum r]
    W: np.ndarray        # [sum r, N]

    @property
    def sum_rank(self):
        return int(self.r.sum())


def all_pairs(O):
    pi, pj = np.triu_indices(O)
    return pi.astype(np.int32), pj.astype(np.int32)


def full_svd_pairs(Lbar, pi, pj):
    """O4 first half: full sorted SVD of the listed pair blocks (OpenMP over pairs)."""
    Lbar = _f64(Lbar)
    X, O, N = Lbar.shape
    pi = np.ascontiguousarray(pi, dtype=np.int32)
    pj = np.ascontiguousarray(pj, dtype=np.int32)
    n = len(pi)
    Ut, s, Wt = np.empty((n, N, N)), np.empty((n, N)), np.empty((n, N, N))
    _l().orc_factor_pairs(C.c_int(N), C.c_int(X), C.c_int(O), _p(Lbar), C.c_int(n), _p(pi), _p(pj), _p(Ut), _p(s), _p(Wt))
    return Ut, s, Wt


def truncate(N, O, pi, pj, Ut, s, Wt, T) -> FactorSet:
    """O4 second half (Eq. 18): keep the K with sigma_K > T (strict, absolute)."""
    r = (s > T).sum(axis=1).astype(np.int32)
    off = np.zeros(len(r), dtype=np.int64)
    off[1:] = np.cumsum(r)[:-1]
    R = int(r.sum())
    U, W, sg = np.empty((R, N)), np.empty((R, N)), np.empty(R)
    for k in range(len(r)):
        U[off[k]:off[k] + r[k]] = Ut[k, :r[k]]
        W[off[k]:off[k] + r[k]] = Wt[k, :r[k]]
        sg[off[k]:off[k] + r[k]] = s[k, :r[k]]
    return FactorSet(N, O, np.asarray(pi, np.int32), np.asarray(pj, np.int32), r, off, U, sg, W)


def own_factors(Lbar, T) -> FactorSet:
    """O4: the oracle's own factor set of one spin at threshold T, all pairs i<=j."""
    X, O, N = Lbar.shape
    pi, pj = all_pairs(O)
    Ut, s, Wt = full_svd_pairs(Lbar, pi, pj)
    return truncate(N, O, pi, pj, Ut, s, Wt, T)


def make_factor_set(N, O, pi, pj, r, U, sigma, W) -> FactorSet:
    """Wrap factors obtained elsewhere (e.g. lo_factor_pair of the library under test) for O5."""
    r = np.ascontiguousarray(r, dtype=np.int32)
    off = np.zeros(len(r), dtype=np.int64)
    off[1:] = np.cumsum(r)[:-1]
    return FactorSet(N, O, np.ascontiguousarray(pi, np.int32), np.ascontiguousarray(pj, np.int32), r, off,
                     _f64(U).reshape(-1, N), _f64(sigma).reshape(-1), _f64(W).reshape(-1, N))


# ------------------------------------------------------------------ NEXT-4: pair screening (section 4)
def pair_norm_bounds(Lbar, pi, pj):
    """Upper bounds on the largest singular value of the pair blocks Y^{ij} = sum_g l^g_i (l^g_j)^T, l^g_i = Lbar[g, i, :]
    (PAPER.md:133), that need no SVD -- the rigorous pre-SVD screen: a pair whose bound is <= T has rank 0 under Eq. 18.
        sigma_1(Y^{ij}) <= |Y^{ij}|_F                      (spectral <= Frobenius norm)
                        <= sum_g |l^g_i|_2 |l^g_j|_2       (triangle inequality over the rank-one terms; keeps the locality
                                                            of every Cholesky vector, so it decays with the distance i-j)
                        <= |Lbar_i|_F |Lbar_j|_F           (Cauchy-Schwarz over g; distance-blind)
    Returns (fro [n], tri [n], cs [n]) for the listed pairs, plain loops."""
    Lbar = _f64(Lbar)
    X, O, N = Lbar.shape
    nrm = np.zeros((X, O))
    for g in range(X):
        for i in range(O):
            nrm[g, i] = np.sqrt((Lbar[g, i] * Lbar[g, i]).sum())
    fro, tri, cs = np.zeros(len(pi)), np.zeros(len(pi)), np.zeros(len(pi))
    for k in range(len(pi)):
        i, j = int(pi[k]), int(pj[k])
        Y = pair_eri(Lbar, i, j)
        fro[k] = np.sqrt((Y * Y).sum())
        t = 0.0
        for g in range(X):
            t += nrm[g, i] * nrm[g, j]
        tri[k] = t
        cs[k] = np.sqrt((nrm[:, i] ** 2).sum()) * np.sqrt((nrm[:, j] ** 2).sum())
    return fro, tri, cs


def screen_pairs(fs: FactorSet, cutoff):
    """Energy screen ("screening pairs of electrons, and only including those that contribute meaningfully to the total
    energy"): pair (i, j) is dropped (rank 0) when  m_ij sigma_1^{ij} <= cutoff,  m_ij = 2 - delta_ij.  Since
    |sum_K sigma_K a_K b_K| = |Theta_j^T Y_r Theta_i| <= sigma_1 |Theta_i|_2 |Theta_j|_2, the exchange energy of a walker moves
    by at most  cK sum_dropped m_ij sigma_1^{ij} |Theta_i|_2 |Theta_j|_2  (cK = 1 closed shell, 1/2 per spin unrestricted).
    Returns (screened FactorSet, dropped [n_pairs] bool, m_ij sigma_1 [n_pairs])."""
    n = len(fs.r)
    ms1 = np.zeros(n)
    drop = np.zeros(n, dtype=bool)
    for k in range(n):
        m = 1.0 if fs.pi[k] == fs.pj[k] else 2.0
        s1 = fs.sigma[fs.off[k]] if fs.r[k] > 0 else 0.0
        ms1[k] = m * s1
        drop[k] = fs.r[k] > 0 and ms1[k] <= cutoff
    r = np.where(drop, 0, fs.r).astype(np.int32)
    rows = [np.arange(fs.off[k], fs.off[k] + r[k]) for k in range(n)]
    rows = np.concatenate(rows) if rows else np.zeros(0, np.int64)
    return make_factor_set(fs.N, fs.O, fs.pi, fs.pj, r, fs.U[rows], fs.sigma[rows], fs.W[rows]), drop, ms1


def randomized_svd(Y, Omega):
    """Approximate SVD of one pair block by a randomised range finder ("approximate versions of the singular value
    decomposition, which would reduce the scaling of this step significantly"; Halko, Martinsson & Tropp
    2011, Alg. 4.1 + 5.1), written out step by step with library primitives as steps:
        Z = Y^T Omega                     sketch of the row space of Y            (Omega: n x k Gaussian test matrix, an INPUT)
        P = orth(Z)                       numpy.linalg.qr
        B = P^T Y^T                       k x n
        B = Ub diag(s) Vb^T               numpy.linalg.svd of the small matrix
        Y ~= Vb diag(s) (P Ub)^T          => left vectors Vb^T rows, right vectors (P Ub)^T rows
        resid = |Y - U^T diag(s) W|_F     a-posteriori error: every singular value of Y is within resid of the returned ones
                                          (Weyl), so the result is exact to working accuracy iff rank(Y) <= k numerically.
    Returns (Ut [k,n], s [k] descending, Wt [k,n], resid)."""
    Y, Omega = _f64(Y), _f64(Omega)
    Z = Y.T @ Omega
    P, _ = np.linalg.qr(Z)
    B = P.T @ Y.T
    Ub, s, Vbt = np.linalg.svd(B, full_matrices=False)
    Ut = Vbt
    Wt = (P @ Ub).T
    resid = float(np.sqrt(((Y - (Ut.T * s) @ Wt) ** 2).sum()))
    return Ut, s, Wt, resid


def _fs_args(fs: FactorSet):
    return (C.c_int(fs.N), C.c_int(fs.O), C.c_int(len(fs.r)), _p(fs.pi), _p(fs.pj), _p(fs.r), _p(fs.off),
            _p(fs.U), _p(fs.sigma), _p(fs.W))


def exchange_lo(fs: FactorSet, th):
    """O5 single-spin truncated exchange sum, Eq. 19/22."""
    th = _c128(th)
    out = np.zeros(1, dtype=np.complex128)
    _l().orc_exchange_lo(*_fs_args(fs), _p(th), _p(out))
    return out[0]


def exchange_lo_batch(fs: FactorSet, thetas):
    """O5 single-spin truncated exchange sums of several walkers (thetas [n_w,N,O]); OpenMP over walkers."""
    thetas = _c128(thetas)
    out = np.zeros(thetas.shape[0], dtype=np.complex128)
    _l().orc_exchange_lo_batch(C.c_int(thetas.shape[0]), *_fs_args(fs), _p(thetas), _p(out))
    return out


def coulomb_lo(fs: FactorSet, th):
    """Paper-literal compressed Coulomb double sum S (closed shell E_J^LO = 2 S), Eq. 19/22."""
    th = _c128(th)
    out = np.zeros(1, dtype=np.complex128)
    _l().orc_coulomb_lo(*_fs_args(fs), _p(th), _p(out))
    return out[0]


# ------------------------------------------------------------------ whole energies
def local_energy_exact(h, L, psis, phis, route="cholesky"):
    """Exact (untruncated) local energy of ONE walker: returns (E_L, E1, E_J, E_K).
    route: 'bruteforce' (O1), 'cholesky' (O2), 'full_eri' (O3).  psis/phis: per-spin lists."""
    ns = len(psis)
    ths = []
    for psi, phi in zip(psis, phis):
        th, _, st = theta(psi, phi)
        if st:
            nan = complex(np.nan, np.nan)
            return nan, nan, nan, nan
        ths.append(th)
    if route == "bruteforce":
        Gs = [green(psi, th) for psi, th in zip(psis, ths)]
        e1, ej, ek = energy_bruteforce(h, L, Gs[0], Gs[1] if ns == 2 else None)
        return e1 + ej + ek, e1, ej, ek
    hr = [half_rotate(L, h, psi) for psi in psis]
    e1, ej = onebody_coulomb([a for a, _ in hr], [b for _, b in hr], ths)
    fn = exchange_cholesky if route == "cholesky" else exchange_full_eri
    ek = sum(fn(hr[s][0], ths[s]) for s in range(ns))
    if ns == 2:
        ek *= 0.5
    return e1 + ej + ek, e1, ej, ek


def local_energy_lo(psis, Lbars, hbars, fsets, phis):
    """The LO local energy of a batch of walkers on given factor sets (one per spin):
    returns (E [n_w,4] = E_L,E1,E_J,E_K ; status [n_w]).  OpenMP over walkers; bench.py's cpu_baseline."""
    ns = len(psis)
    psis = [_f64(a) for a in psis]
    Lbars = [_f64(a) for a in Lbars]
    hbars = [_f64(a) for a in hbars]
    phis = [_c128(a) for a in phis]
    n_w, N, _ = phis[0].shape
    X = Lbars[0].shape[0]
    O = (C.c_int * ns)(*[a.shape[1] for a in psis])
    npairs = (C.c_int * ns)(*[len(f.r) for f in fsets])
    out = np.zeros((n_w, 4), dtype=np.complex128)
    status = np.zeros(n_w, dtype=np.int32)
    _l().orc_local_energy_lo(C.c_int(n_w), C.c_int(N), C.c_int(X), C.c_int(ns), O, _ptr_array(psis), _ptr_array(Lbars),
                             _ptr_array(hbars), npairs, _ptr_array([f.pi for f in fsets]), _ptr_array([f.pj for f in fsets]),
                             _ptr_array([f.r for f in fsets]), _ptr_array([f.off for f in fsets]),
                             _ptr_array([f.U for f in fsets]), _ptr_array([f.sigma for f in fsets]),
                             _ptr_array([f.W for f in fsets]), _ptr_array(phis), _p(out), _p(status))
    return out, status


def empty_factor_set(N, O) -> FactorSet:
    z = np.zeros(0, np.int32)
    return FactorSet(N, O, z, z, z, np.zeros(0, np.int64), np.zeros((0, N)), np.zeros(0), np.zeros((0, N)))


def local_energy_lo_streamed(psis, Lbars, hbars, phis, n_pairs, fetch, chunk=256):
    """local_energy_lo for factor sets too large to hold on the host: Theta, E1 and E_J as in local_energy_lo, the
    exchange sum accumulated over chunks of pairs, fetch(spin, k0, k1) -> FactorSet of the pairs [k0, k1) of that spin
    (natural i<=j order).  Returns (E [n_w,4], status [n_w], seconds spent in the oracle's own arithmetic)."""
    import time
    ns = len(psis)
    t0 = time.time()
    E, status = local_energy_lo(psis, Lbars, hbars, [empty_factor_set(p.shape[0], p.shape[1]) for p in psis], phis)
    n_w = phis[0].shape[0]
    thetas = []
    for s in range(ns):
        th = np.zeros(phis[s].shape, dtype=np.complex128)
        for w in range(n_w):
            if status[w] == 0:
                th[w] = theta(psis[s], phis[s][w])[0]
        thetas.append(th)
    secs = time.time() - t0
    ek = np.zeros(n_w, dtype=np.complex128)
    for s in range(ns):
        for k0 in range(0, n_pairs[s], chunk):
            fs = fetch(s, k0, min(n_pairs[s], k0 + chunk))
            t0 = time.time()
            ek += exchange_lo_batch(fs, thetas[s])
            secs += time.time() - t0
    if ns == 2:
        ek *= 0.5
    ok = status == 0
    E[ok, 3] = ek[ok]
    E[ok, 0] = E[ok, 1] + E[ok, 2] + E[ok, 3]
    return E, status, secs


# ------------------------------------------------------------------ NEXT-2: multi-determinant trial (Eq. 12, 13)
def sub_factor_set(fs: FactorSet, cols) -> FactorSet:
    """Factors of the pairs among the orbitals `cols` (ascending) of a factor set over more orbitals, re-indexed to
    0..len(cols)-1: the integrals of a determinant that occupies exactly those orbitals."""
    cols = np.asarray(cols)
    assert (np.diff(cols) > 0).all()
    pos = -np.ones(fs.O, dtype=np.int64)
    pos[cols] = np.arange(len(cols))
    keep = [k for k in range(len(fs.r)) if pos[fs.pi[k]] >= 0 and pos[fs.pj[k]] >= 0]
    rows = np.concatenate([np.arange(fs.off[k], fs.off[k] + fs.r[k]) for k in keep]) if keep else np.zeros(0, np.int64)
    return make_factor_set(fs.N, len(cols), pos[fs.pi[keep]], pos[fs.pj[keep]], fs.r[keep], fs.U[rows], fs.sigma[rows], fs.W[rows])


def local_energy_cas(Cmo, columns, coef, Lbar, hbar, fs, phi, exact=False, compressed_coulomb=False):
    """Local energy of ONE closed-shell walker phi [N,O] with the multi-determinant trial sum_d c_d |d>, every |d> a
    closed-shell determinant occupying the orbitals columns[d] (columns of Cmo, in the reference's column positions),
    straight from the definition (Eq. 12 with Eq. 13, applied to every energy term):
        E = sum_d w_d E^d / sum_d w_d,   w_d = c_d <d|phi> = c_d det(Psi_d^T phi)^2   (alpha and beta strings equal),
    E^d = the single-determinant local energy with trial Psi_d = Cmo[:, columns[d]] (Theta^d by its own LU, Eq. 15).
    Lbar [X,n_orb,N], hbar [n_orb,N]: half-rotated integrals for ALL orbitals of Cmo; fs: factor set over all their
    pairs (exchange by O5 on the sub-set of pairs the determinant occupies); exact=True uses the Cholesky route (O2)
    for the exchange instead; compressed_coulomb=True takes E_J from the factors too (Eq. 19/22 first term, the paper's
    own multi-determinant expression Eq. 22).  Returns (E_L, E1, E_J, E_K, sum_d w_d / det(Psi_0^T phi)^2)."""
    Cmo, phi = _f64(Cmo), _c128(phi)
    num = np.zeros(3, dtype=np.complex128)
    den = 0.0 + 0.0j
    w0 = None
    for d, cols in enumerate(columns):
        cols = np.asarray(cols)
        th, det, st = theta(Cmo[:, cols], phi)
        if w0 is None:
            w0 = det * det                    # determinant 0 is the reference
        if st != 0:
            continue                          # <d|phi> = 0: no contribution
        order = np.argsort(cols)
        sc = cols[order]
        ths = np.ascontiguousarray(th[:, order])
        e1, ej = onebody_coulomb([np.ascontiguousarray(Lbar[:, sc, :])], [np.ascontiguousarray(hbar[sc])], [ths])
        ek = exchange_cholesky(np.ascontiguousarray(Lbar[:, sc, :]), ths) if exact else exchange_lo(sub_factor_set(fs, sc), ths)
        if compressed_coulomb:
            ej = 2.0 * coulomb_lo(sub_factor_set(fs, sc), ths)
        w = coef[d] * det * det
        num += w * np.array([e1, ej, ek])
        den += w
    E = num / den
    return E.sum(), E[0], E[1], E[2], den / w0


def local_energy_cas_u(Cmo, columns, coef, Lbar, hbar, fs, phi):
    """Unrestricted version of local_energy_cas: per-spin lists Cmo[s], columns[s][d], Lbar[s], hbar[s], fs[s], phi[s];
    determinant d = |alpha string d>|beta string d>, w_d = c_d det(Psi_d^a^T phi_a) det(Psi_d^b^T phi_b), and E^d by the
    unrestricted formulas (E1 summed over spins, E_J = 1/2 sum_g (X_a+X_b)^2, E_K = 1/2 sum over same-spin
    pairs).  Returns (E_L, E1, E_J, E_K, sum_d w_d / w_reference)."""
    num = np.zeros(3, dtype=np.complex128)
    den = 0.0 + 0.0j
    w0 = None
    for d in range(len(coef)):
        ths, Ls, hs, dets, ek, bad = [], [], [], [], 0.0 + 0.0j, False
        for s in range(2):
            cols = np.asarray(columns[s][d])
            th, det, st = theta(_f64(Cmo[s])[:, cols], _c128(phi[s]))
            bad |= st != 0
            order = np.argsort(cols)
            sc = cols[order]
            t = np.ascontiguousarray(th[:, order])
            ths.append(t)
            Ls.append(np.ascontiguousarray(Lbar[s][:, sc, :]))
            hs.append(np.ascontiguousarray(hbar[s][sc]))
            dets.append(det)
            if not bad:
                ek += 0.5 * exchange_lo(sub_factor_set(fs[s], sc), t)
        if w0 is None:
            w0 = dets[0] * dets[1]
        if bad:
            continue
        e1, ej = onebody_coulomb(Ls, hs, ths)
        w = coef[d] * dets[0] * dets[1]
        num += w * np.array([e1, ej, ek])
        den += w
    E = num / den
    return E.sum(), E[0], E[1], E[2], den / w0
