"""Pins of the CPU oracle: the oracle is checked against what the paper and the
mathematics fix -- four algebraically equal routes (Eq. 10/16/17/19 at T=0), the closed-form HF energy,
invariances, projector identities, degenerate cases, Eckart-Young, the truncation bound, textbook SVDs and
numpy's LAPACK SVD.  CPU only."""
import math

import numpy as np
import pytest

import gen
import oracle

RTOL = 1e-11


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def exact(P, phis, w, route):
    return np.array(oracle.local_energy_exact(P.h, P.L, P.psi, [ph[w] for ph in phis], route))


# ---------------------------------------------------------------- P1 / P2: four routes agree at T=0
def test_p1_routes_agree_c0(c0, c0_walkers):
    Lbar, hbar = oracle.half_rotate(c0.L, c0.h, c0.psi[0])
    fs0 = oracle.own_factors(Lbar, 0.0)
    assert (fs0.r == c0.N).all()                      # T=0 keeps every sigma>0
    E_lo, st = oracle.local_energy_lo(c0.psi, [Lbar], [hbar], [fs0], c0_walkers)
    assert (st == 0).all()
    for w in range(c0.n_w):
        e_bf = exact(c0, c0_walkers, w, "bruteforce")     # Eq. 10
        e_ch = exact(c0, c0_walkers, w, "cholesky")       # Eq. 16
        e_fe = exact(c0, c0_walkers, w, "full_eri")       # Eq. 17
        scale = abs(e_bf[0])
        for k in range(4):
            assert abs(e_ch[k] - e_bf[k]) <= RTOL * max(scale, abs(e_bf[k]))
            assert abs(e_fe[k] - e_bf[k]) <= RTOL * max(scale, abs(e_bf[k]))
            assert abs(E_lo[w, k] - e_bf[k]) <= RTOL * max(scale, abs(e_bf[k]))   # Eq. 19 at T=0


def test_p2_untruncated_svd_exact_c1(c1, c1_walkers):
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, c1.psi[0])
    fs0 = oracle.own_factors(Lbar, 0.0)
    E_lo, _ = oracle.local_energy_lo(c1.psi, [Lbar], [hbar], [fs0], [c1_walkers[0][:3]])
    for w in range(3):
        th, _, _ = oracle.theta(c1.psi[0], c1_walkers[0][w])
        ek = oracle.exchange_cholesky(Lbar, th)
        assert abs(E_lo[w, 3] - ek) <= 1e-11 * abs(ek)
        assert abs(oracle.exchange_full_eri(Lbar, th) - ek) <= 1e-11 * abs(ek)


# ---------------------------------------------------------------- P3: closed-form HF energy
@pytest.mark.parametrize("cfg", ["c0", "c1"])
def test_p3_hf_closed_form(cfg, request):
    P = request.getfixturevalue(cfg)
    psi = P.psi[0]
    D = psi @ psi.T
    LD = np.einsum("gpq,qr->gpr", P.L, D)
    e_hf = 2 * np.trace(P.h @ D) + 2 * (np.trace(LD, axis1=1, axis2=2) ** 2).sum() - np.einsum("gpr,grp->", LD, LD)
    routes = ["bruteforce", "cholesky", "full_eri"] if cfg == "c0" else ["cholesky", "full_eri"]
    for route in routes:
        e = oracle.local_energy_exact(P.h, P.L, P.psi, [psi.astype(np.complex128)], route)[0]
        assert e.imag == 0.0
        assert rel(e.real, e_hf) < 1e-11
    th, det, st = oracle.theta(psi, psi.astype(np.complex128))
    assert st == 0 and np.abs(th - psi).max() < 1e-13 and abs(det - 1) < 1e-12


# ---------------------------------------------------------------- P4: occupied rotation
def test_p4_occupied_rotation(c1, c1_walkers):
    psi = c1.psi[0]
    R = gen.random_orthogonal(psi.shape[1], 7)
    psi_r = psi @ R
    phi = c1_walkers[0][1]
    e0 = np.array(oracle.local_energy_exact(c1.h, c1.L, [psi], [phi], "cholesky"))
    e1 = np.array(oracle.local_energy_exact(c1.h, c1.L, [psi_r], [phi], "cholesky"))
    assert np.abs(e0 - e1).max() <= 1e-10 * abs(e0[0])
    # LO at T=0 with the rotated (delocalised) trial is still exact
    Lb_r, hb_r = oracle.half_rotate(c1.L, c1.h, psi_r)
    pi, pj = np.array([0, 0, 3], np.int32), np.array([0, 5, 17], np.int32)
    Ut, s, Wt = oracle.full_svd_pairs(Lb_r, pi, pj)
    th, _, _ = oracle.theta(psi_r, phi)
    for k in range(3):
        Y = oracle.pair_eri(Lb_r, pi[k], pj[k])
        exact_e = th[:, pj[k]] @ Y @ th[:, pi[k]]
        lo = ((Ut[k] @ th[:, pj[k]]) * s[k] * (Wt[k] @ th[:, pi[k]])).sum()
        assert abs(lo - exact_e) <= 1e-11 * abs(exact_e)


def test_p4_localised_compresses_better():
    # delocalising the trial raises the ranks at fixed T>0.  Use the rank-structured
    # "vector" reading where distance decay drives the ranks.
    P = gen.make_problem(1, reading="vector")
    psi = P.psi[0]
    Lb, _ = oracle.half_rotate(P.L, P.h, psi)
    Lb_r, _ = oracle.half_rotate(P.L, P.h, psi @ gen.random_orthogonal(psi.shape[1], 3))
    pi, pj = oracle.all_pairs(psi.shape[1])
    sel = slice(0, None, 7)
    _, s, _ = oracle.full_svd_pairs(Lb, pi[sel], pj[sel])
    _, s_r, _ = oracle.full_svd_pairs(Lb_r, pi[sel], pj[sel])
    T = 1e-2
    assert (s_r > T).sum() > (s > T).sum()


# ---------------------------------------------------------------- P5: walker gauge invariance
def test_p5_gauge(c0, c0_walkers):
    rng = np.random.default_rng(5)
    O = c0.n_occ[0]
    Cm = rng.standard_normal((O, O)) + 1j * rng.standard_normal((O, O))
    phi = c0_walkers[0][2]
    e0 = np.array(oracle.local_energy_exact(c0.h, c0.L, c0.psi, [phi], "cholesky"))
    e1 = np.array(oracle.local_energy_exact(c0.h, c0.L, c0.psi, [phi @ Cm], "cholesky"))
    assert np.abs(e0 - e1).max() <= 1e-9 * abs(e0[0]) * np.linalg.cond(Cm)


# ---------------------------------------------------------------- P6: projector identities
@pytest.mark.parametrize("cfg", ["c0", "c1"])
def test_p6_projector(cfg, request):
    P = request.getfixturevalue(cfg)
    W = request.getfixturevalue(cfg + "_walkers")
    psi, phi = P.psi[0], W[0][0]
    th, det, st = oracle.theta(psi, phi)
    O = psi.shape[1]
    assert st == 0
    assert np.abs(psi.T @ th - np.eye(O)).max() < 1e-11
    G = oracle.green(psi, th)
    assert abs(np.trace(G) - O) < 1e-10
    assert np.abs(G @ G - G).max() < 1e-10
    assert rel(det, np.linalg.det(psi.T @ phi)) < 1e-11
    assert np.abs(th - phi @ np.linalg.inv(psi.T @ phi)).max() < 1e-10       # library routine (LAPACK)


def test_singular_overlap_flagged(c0):
    psi = c0.psi[0]
    phi = psi.astype(np.complex128).copy()
    phi[:, 1] = phi[:, 0]
    _, _, st = oracle.theta(psi, phi)
    assert st == 1


# ---------------------------------------------------------------- P7: degenerate cases
def test_p7_single_orbital():
    xyz, fns = gen.site_geometry(0)
    P = gen.make_problem_from_geometry(xyz, fns, (1,), 40, seed=11)
    phi = gen.make_walkers(P, 3)[0]
    for w in range(3):
        _, _, ej, ek = oracle.local_energy_exact(P.h, P.L, P.psi, [phi[w]], "cholesky")
        assert abs(ek + ej / 2) <= 1e-12 * abs(ej)


def test_p7_single_cholesky_vector():
    xyz, fns = gen.site_geometry(0)
    P = gen.make_problem_from_geometry(xyz, fns, (4,), 1, seed=12)
    Lbar, hbar = oracle.half_rotate(P.L, P.h, P.psi[0])
    pi, pj = oracle.all_pairs(4)
    Ut, s, Wt = oracle.full_svd_pairs(Lbar, pi, pj)
    assert (s[:, 1] <= 1e-12 * s[:, 0]).all()                 # every Y^{ij} has rank <= 1
    fs = oracle.truncate(P.N, 4, pi, pj, Ut, s, Wt, 0.5 * s[:, 0].min())
    assert (fs.r == 1).all()
    phi = gen.make_walkers(P, 2)
    E, _ = oracle.local_energy_lo(P.psi, [Lbar], [hbar], [fs], phi)
    for w in range(2):
        e = oracle.local_energy_exact(P.h, P.L, P.psi, [phi[0][w]], "bruteforce")
        assert abs(E[w, 3] - e[3]) <= 1e-12 * abs(e[3])


# ---------------------------------------------------------------- P8: Eckart-Young, orthonormality, monotone ranks, bound
def test_p8_eckart_young_and_bound(c1, c1_walkers):
    psi = c1.psi[0]
    O, N = psi.shape[1], c1.N
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, psi)
    pi, pj = oracle.all_pairs(O)
    Ut, s, Wt = oracle.full_svd_pairs(Lbar, pi, pj)
    assert (np.diff(s, axis=1) <= 0).all()
    for k in (0, 5, 100, len(pi) - 1):
        assert np.abs(Ut[k] @ Ut[k].T - np.eye(N)).max() < 1e-12
        assert np.abs(Wt[k] @ Wt[k].T - np.eye(N)).max() < 1e-12
        Y = oracle.pair_eri(Lbar, pi[k], pj[k])
        for r in (0, 3, N // 2, N):
            err2 = np.linalg.norm(Y - (Ut[k, :r].T * s[k, :r]) @ Wt[k, :r]) ** 2
            assert abs(err2 - (s[k, r:] ** 2).sum()) <= 1e-10 * (s[k] ** 2).sum()
    ranks = [int((s > T).sum()) for T in (0.0, 1e-6, 1e-4, 1e-2, 1.0, 10.0)]
    assert all(a >= b for a, b in zip(ranks, ranks[1:])) and ranks[0] > ranks[-1]
    # truncation bound: |E_K^LO - E_K| <= sum_{i<=j} m_ij sigma_{r+1} |Theta_i| |Theta_j|
    m = np.where(pi == pj, 1.0, 2.0)
    for T in (1.0, 5.0):
        fs = oracle.truncate(N, O, pi, pj, Ut, s, Wt, T)
        assert 0 < fs.sum_rank < N * len(pi)
        for w in range(2):
            th, _, _ = oracle.theta(psi, c1_walkers[0][w])
            nrm = np.linalg.norm(th, axis=0)
            s_next = np.array([s[k, fs.r[k]] if fs.r[k] < N else 0.0 for k in range(len(pi))])
            bound = (m * s_next * nrm[pi] * nrm[pj]).sum()
            err = abs(oracle.exchange_lo(fs, th) - oracle.exchange_cholesky(Lbar, th))
            assert 0 < err <= bound <= T * nrm.sum() ** 2


# ---------------------------------------------------------------- P9: real walkers, unrestricted = closed shell
def test_p9_real_walker_real_energy(c0):
    phi = gen.make_walkers(c0, 2, real=True)
    for route in ("bruteforce", "cholesky", "full_eri"):
        e = oracle.local_energy_exact(c0.h, c0.L, c0.psi, [phi[0][0]], route)
        assert all(x.imag == 0.0 for x in e)


def test_p9_unrestricted_equals_closed_shell(c0, c0_walkers):
    phi = c0_walkers[0][3]
    for route in ("bruteforce", "cholesky", "full_eri"):
        e_r = np.array(oracle.local_energy_exact(c0.h, c0.L, c0.psi, [phi], route))
        e_u = np.array(oracle.local_energy_exact(c0.h, c0.L, [c0.psi[0], c0.psi[0]], [phi, phi], route))
        assert np.abs(e_r - e_u).max() <= 1e-12 * np.abs(e_r).max()


def test_o6_unrestricted_routes_agree():
    xyz, fns = gen.site_geometry(0)
    P = gen.make_problem_from_geometry(xyz, fns, (5, 3), 60, seed=21)
    phis = gen.make_walkers(P, 3)
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]
    fsets = [oracle.own_factors(a, 0.0) for a, _ in hr]
    E, st = oracle.local_energy_lo(P.psi, [a for a, _ in hr], [b for _, b in hr], fsets, phis)
    for w in range(3):
        ph = [phis[0][w], phis[1][w]]
        e_bf = np.array(oracle.local_energy_exact(P.h, P.L, P.psi, ph, "bruteforce"))
        for route in ("cholesky", "full_eri"):
            e = np.array(oracle.local_energy_exact(P.h, P.L, P.psi, ph, route))
            assert np.abs(e - e_bf).max() <= 1e-11 * np.abs(e_bf).max()
        assert np.abs(E[w] - e_bf).max() <= 1e-11 * np.abs(e_bf).max()


# ---------------------------------------------------------------- P10: the Jacobi SVD itself
def hilbert(n):
    i = np.arange(n)
    return 1.0 / (i[:, None] + i[None, :] + 1.0)


def test_p10_svd_diagonal_and_rank1():
    d = np.array([3.0, 0.5, 7.0, 1e-3, 2.0])
    Ut, s, Wt = oracle.svd(np.diag(d))
    assert np.allclose(s, np.sort(d)[::-1], rtol=1e-15)
    u, v = np.arange(1.0, 7.0), np.array([1.0, -2.0, 0.5, 3.0, 0.0, 1.0])
    Ut, s, Wt = oracle.svd(np.outer(u, v))
    assert rel(s[0], np.linalg.norm(u) * np.linalg.norm(v)) < 1e-14 and (s[1:] < 1e-13).all()
    assert np.abs(np.abs(Ut[0]) - u / np.linalg.norm(u)).max() < 1e-14
    assert np.abs(np.abs(Wt[0]) - np.abs(v) / np.linalg.norm(v)).max() < 1e-14
    Ut, s, Wt = oracle.svd(np.zeros((4, 4)))
    assert (s == 0).all()


@pytest.mark.parametrize("n", [3, 5, 8])
def test_p10_svd_hilbert(n):
    # Hilbert matrix: SPD, so singular values = eigenvalues; sum = trace = sum 1/(2i-1),
    # product = det(H_n) = c_n^4 / c_{2n}, c_n = prod_{i<n} i!  (textbook closed forms)
    H = hilbert(n)
    Ut, s, Wt = oracle.svd(H)
    assert rel(s.sum(), sum(1.0 / (2 * i + 1) for i in range(n))) < 1e-14
    c = lambda m: math.prod(math.factorial(i) for i in range(1, m))
    det = c(n) ** 4 / c(2 * n)
    assert rel(np.prod(s), det) < 1e-12 * np.linalg.cond(H) ** 0.5
    s_np = np.linalg.svd(H, compute_uv=False)
    assert np.abs(s - s_np).max() <= 1e-15 * s[0] * n
    assert (np.abs(s - s_np) <= 1e-10 * s_np + 4e-16 * s[0]).all()    # LAPACK's small sigmas are only abs-accurate
    assert np.abs((Ut.T * s) @ Wt - H).max() < 1e-15 * n


def test_p10_svd_vs_lapack_random_and_pair_block(c1):
    rng = np.random.default_rng(0)
    A = rng.standard_normal((40, 40)) * np.exp(-0.3 * np.arange(40))[None, :]
    Lbar, _ = oracle.half_rotate(c1.L, c1.h, c1.psi[0])
    for M in (A, oracle.pair_eri(Lbar, 2, 9)):
        Ut, s, Wt = oracle.svd(M)
        s_np = np.linalg.svd(M, compute_uv=False)
        assert np.abs(s - s_np).max() <= 1e-13 * s_np[0]
        assert np.abs((Ut.T * s) @ Wt - M).max() <= 1e-13 * s_np[0]
        assert np.abs(Ut @ Ut.T - np.eye(len(s))).max() < 1e-12


def test_pair_eri_symmetry_and_definition(c0):
    Lbar, hbar = oracle.half_rotate(c0.L, c0.h, c0.psi[0])
    assert np.abs(Lbar - np.einsum("gpq,qi->gip", c0.L, c0.psi[0])).max() < 1e-12
    assert np.abs(hbar - c0.psi[0].T @ c0.h).max() < 1e-12
    Y = oracle.pair_eri(Lbar, 1, 4)
    assert np.abs(Y - oracle.pair_eri(Lbar, 4, 1).T).max() == 0.0                         # Y^{ji} = (Y^{ij})^T
    assert np.abs(Y - np.einsum("gp,gq->pq", Lbar[:, 1], Lbar[:, 4])).max() < 1e-11


# ---------------------------------------------------------------- D9: paper-literal compressed Coulomb
def test_coulomb_lo_equals_cholesky_route_at_t0(c0, c0_walkers):
    Lbar, hbar = oracle.half_rotate(c0.L, c0.h, c0.psi[0])
    fs0 = oracle.own_factors(Lbar, 0.0)
    th, _, _ = oracle.theta(c0.psi[0], c0_walkers[0][0])
    _, ej = oracle.onebody_coulomb([Lbar], [hbar], [th])
    assert abs(2 * oracle.coulomb_lo(fs0, th) - ej) <= 1e-11 * abs(ej)


# ---------------------------------------------------------------- regression anchor (written by tests/golden/make_golden.py)
def test_golden_c0_regression(c0, c0_walkers):
    import os
    ref = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "c0_exact_energies.txt"))
    for w in range(c0.n_w):
        e = exact(c0, c0_walkers, w, "cholesky")
        got = np.array([x for z in e for x in (z.real, z.imag)])
        assert np.abs(got - ref[w]).max() <= 1e-11 * np.abs(ref[w]).max()


def test_streamed_evaluation_equals_one_piece(c1, c1_walkers):
    """local_energy_lo_streamed (chunks of pairs, used for the factor sets too large for the host) adds up to
    local_energy_lo on the same factors."""
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, c1.psi[0])
    pi, pj = oracle.all_pairs(c1.n_occ[0])
    sel = np.arange(0, len(pi), 7)
    Ut, s, Wt = oracle.full_svd_pairs(Lbar, pi[sel], pj[sel])
    fs = oracle.truncate(c1.N, c1.n_occ[0], pi[sel], pj[sel], Ut, s, Wt, 1e-2)
    phis = [c1_walkers[0][:5]]
    E, st = oracle.local_energy_lo(c1.psi, [Lbar], [hbar], [fs], phis)

    def fetch(spin, k0, k1):
        r = fs.r[k0:k1]
        a, b = int(fs.off[k0]), int(fs.off[k0] + r.sum())
        return oracle.make_factor_set(c1.N, c1.n_occ[0], fs.pi[k0:k1], fs.pj[k0:k1], r, fs.U[a:b], fs.sigma[a:b], fs.W[a:b])

    Es, sts, secs = oracle.local_energy_lo_streamed(c1.psi, [Lbar], [hbar], phis, [len(sel)], fetch, chunk=5)
    assert (st == 0).all() and (sts == 0).all() and secs > 0
    assert np.abs(Es - E).max() <= 1e-12 * np.abs(E[:, 0]).max()


# ------------------------------------------------------------------------------------------ NEXT-1: propagator
def test_propagator_pins(c0, c0_walkers):
    """B = sum_g x_g L^g.  Pins: a unit field returns that Cholesky matrix exactly; B is symmetric;
    tr B = sum_g x_g tr L^g; and contracting B with the walker's Green's function gives sum_g x_g X^g with the X^g of
    the (already pinned) Coulomb route: sum_pq B_pq G_pq = sum_g x_g sum_ip Lbar^g_ip Theta_pi (Eq. 14, 16)."""
    L, N, X = c0.L, c0.N, c0.n_chol
    for g in (0, 17, X - 1):
        e = np.zeros(X, dtype=np.complex128)
        e[g] = 1.0
        assert np.array_equal(oracle.propagator(L, e), L[g].astype(np.complex128))
    rng = np.random.default_rng(5)
    x = rng.standard_normal(X) + 1j * rng.standard_normal(X)
    B = oracle.propagator(L, x)
    assert np.abs(B - B.T).max() <= 1e-14 * np.abs(B).max()
    tr = sum(x[g] * np.trace(L[g]) for g in range(X))
    assert abs(np.trace(B) - tr) <= 1e-12 * abs(tr)
    psi = c0.psi[0]
    th, _, _ = oracle.theta(psi, c0_walkers[0][0])
    G = oracle.green(psi, th)
    Lbar, hbar = oracle.half_rotate(L, c0.h, psi)
    _, _, Xg = oracle.onebody_coulomb([Lbar], [hbar], [th], want_X=True)
    lhs = (B * G).sum()
    rhs = (x * Xg).sum()
    assert abs(lhs - rhs) <= 1e-12 * abs(rhs)
    # linearity in the fields
    y = rng.standard_normal(X) + 1j * rng.standard_normal(X)
    assert np.abs(oracle.propagator(L, 2.0 * x - 1j * y) - (2.0 * B - 1j * oracle.propagator(L, y))).max() <= 1e-12 * np.abs(B).max()


# ------------------------------------------------------------------------------------------ NEXT-2: multi-determinant trial
def test_cas_exact_eigenstate_two_orbitals():
    """Textbook pin (two electrons in two orbitals of different symmetry): with h diagonal and every Cholesky matrix
    either diagonal or purely off-diagonal, the closed-shell determinants |1 1bar>, |2 2bar> decouple from the singly
    excited ones, H restricted to them is [[2h1+(11|11), (12|12)], [(12|12), 2h2+(22|22)]] (Slater-Condon), and its
    eigenvectors are eigenstates of the full H.  The mixed estimator <Psi_T|H|phi>/<Psi_T|phi> of an eigenstate is its
    eigenvalue for ANY walker: pins the weights c_d det^2, the per-determinant Green's functions and all three terms."""
    h = np.diag([-1.3, 0.4])
    L = np.zeros((3, 2, 2))
    L[0] = np.diag([0.9, 0.5])
    L[1] = np.diag([-0.3, 0.7])
    L[2] = np.array([[0.0, 0.6], [0.6, 0.0]])
    J11, J22, K12 = (L[:2, 0, 0] ** 2).sum(), (L[:2, 1, 1] ** 2).sum(), L[2, 0, 1] ** 2
    H = np.array([[2 * h[0, 0] + J11, K12], [K12, 2 * h[1, 1] + J22]])
    ev, vec = np.linalg.eigh(H)
    Cmo = np.eye(2)
    Lbar, hbar = oracle.half_rotate(L, h, Cmo)
    fs = oracle.own_factors(Lbar, 0.0)
    rng = np.random.default_rng(3)
    for k in range(2):
        for _ in range(3):
            phi = (rng.standard_normal((2, 1)) + 1j * rng.standard_normal((2, 1)))
            for exact in (True, False):
                E = oracle.local_energy_cas(Cmo, [[0], [1]], vec[:, k], Lbar, hbar, fs, phi, exact=exact)
                assert abs(E[0] - ev[k]) <= 1e-12 * max(1.0, abs(ev[k]))


def test_cas_single_determinant_and_bruteforce(c0, c0_walkers):
    """N_det = 1 is the single-determinant energy; a duplicated determinant changes nothing; and for a real expansion
    the weighted sum of per-determinant brute-force energies (Eq. 10 with the G^d of Eq. 13, N^4 sums) agrees."""
    T = gen.make_cas_trial(c0, n_virt=3, n_act_occ=3, n_det=6, max_exc=2)
    Lbar, hbar = oracle.half_rotate(c0.L, c0.h, T.C)
    fs = oracle.own_factors(Lbar, 0.0)
    cols = [T.columns(d) for d in range(T.n_det)]
    phi = c0_walkers[0][1]
    single = oracle.local_energy_exact(c0.h, c0.L, c0.psi, [phi], "cholesky")
    one = oracle.local_energy_cas(T.C, cols[:1], T.coef[:1], Lbar, hbar, fs, phi)
    assert abs(one[0] - single[0]) <= 1e-11 * abs(single[0]) and abs(one[4] - 1.0) <= 1e-13
    dup = oracle.local_energy_cas(T.C, [cols[0], cols[0]], [0.3, 0.9], Lbar, hbar, fs, phi)
    assert abs(dup[0] - single[0]) <= 1e-11 * abs(single[0])
    E = oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi)
    Ex = oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi, exact=True)
    num, den = 0.0, 0.0
    for d in range(T.n_det):
        psi_d = np.ascontiguousarray(T.C[:, cols[d]])
        th, det, st = oracle.theta(psi_d, phi)
        G = oracle.green(psi_d, th)
        e = oracle.energy_bruteforce(c0.h, c0.L, G)
        num += T.coef[d] * det * det * e.sum()
        den += T.coef[d] * det * det
    assert abs(E[0] - num / den) <= 1e-10 * abs(E[0]) and abs(Ex[0] - num / den) <= 1e-10 * abs(E[0])
    assert abs(E[0] - single[0]) > 1e-6 * abs(E[0])          # the expansion does change the energy


def test_cas_unrestricted_pins(c0, c0_walkers):
    """Unrestricted multi-determinant oracle: identical alpha/beta orbitals, strings and walkers reproduce the
    closed-shell multi-determinant energy; one determinant reproduces the unrestricted single-determinant energy."""
    T = gen.make_cas_trial(c0, n_virt=3, n_act_occ=3, n_det=6, max_exc=2)
    Lbar, hbar = oracle.half_rotate(c0.L, c0.h, T.C)
    fs = oracle.own_factors(Lbar, 0.0)
    cols = [T.columns(d) for d in range(T.n_det)]
    phi = c0_walkers[0][2]
    Ec = oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi)
    Eu = oracle.local_energy_cas_u([T.C, T.C], [cols, cols], T.coef, [Lbar, Lbar], [hbar, hbar], [fs, fs], [phi, phi])
    assert np.abs(np.array(Eu) - np.array(Ec)).max() <= 1e-11 * abs(Ec[0])
    # different strings and walkers per spin, one determinant: the unrestricted single-determinant energy
    xyz, fns = gen.site_geometry(0)
    P = gen.make_problem_from_geometry(xyz, fns, (4, 3), 48, seed=5)
    phis = gen.make_walkers(P, 2)
    Ta, Tb = gen.make_cas_trial(P, 2, 2, 4, 2, spin=0), gen.make_cas_trial(P, 2, 2, 4, 2, spin=1)
    hr = [oracle.half_rotate(P.L, P.h, t.C) for t in (Ta, Tb)]
    fss = [oracle.own_factors(a, 0.0) for a, _ in hr]
    colsu = [[Ta.columns(d) for d in range(4)], [Tb.columns(d) for d in range(4)]]
    E1 = oracle.local_energy_cas_u([Ta.C, Tb.C], [colsu[0][:1], colsu[1][:1]], Ta.coef[:1], [a for a, _ in hr], [b for _, b in hr], fss,
                                   [phis[0][1], phis[1][1]])
    Es = oracle.local_energy_exact(P.h, P.L, P.psi, [phis[0][1], phis[1][1]], "cholesky")
    assert np.abs(np.array(E1[:4]) - np.array(Es)).max() <= 1e-10 * abs(Es[0])
    Eall = oracle.local_energy_cas_u([Ta.C, Tb.C], colsu, Ta.coef, [a for a, _ in hr], [b for _, b in hr], fss, [phis[0][1], phis[1][1]])
    assert abs(Eall[0] - Es[0]) > 1e-6 * abs(Es[0])


def test_cas_unrestricted_open_shell_singlet_and_triplet():
    """Pin of oracle.local_energy_cas_u for determinants whose alpha and beta strings DIFFER (Eq. 12/13, PAPER.md:108-114;
    Slater-Condon rules).  One alpha and one beta electron in two orbitals of different symmetry (h diagonal, every
    Cholesky matrix either diagonal or purely off-diagonal): |1a 2b> and |2a 1b> decouple from the closed-shell
    determinants (<1a1b|H|1a2b> = h_12 + (11|12) = 0) and couple to each other through (12|21) = K12, so
        singlet (|1a2b> + |2a1b>)/sqrt2 :  E = h1 + h2 + J12 + K12,
        triplet (|1a2b> - |2a1b>)/sqrt2 :  E = h1 + h2 + J12 - K12,      J12 = sum_g L^g_11 L^g_22,  K12 = sum_g (L^g_12)^2
    are exact eigenstates, and the mixed estimator returns the eigenvalue for ANY pair of alpha/beta walkers.  This
    fixes the weight w_d = c_d det_a det_b (det_a^2 would give another number: det_a != det_b here) and the relative
    sign of determinants with different strings (a flipped coefficient turns the singlet into the triplet, 2 K12 away)."""
    h = np.diag([-0.8, 0.35])
    L = np.zeros((4, 2, 2))
    L[0] = np.diag([0.7, 0.4])
    L[1] = np.diag([-0.2, 0.9])
    L[2] = np.array([[0.0, 0.55], [0.55, 0.0]])
    L[3] = np.array([[0.0, -0.3], [-0.3, 0.0]])
    J12 = (L[:, 0, 0] * L[:, 1, 1]).sum()
    K12 = (L[:, 0, 1] ** 2).sum()
    assert K12 > 0.1
    Cmo = np.eye(2)
    Lbar, hbar = oracle.half_rotate(L, h, Cmo)
    fs = oracle.own_factors(Lbar, 0.0)
    cols = [[[0], [1]], [[1], [0]]]          # alpha strings of the two determinants, beta strings of the two determinants
    rng = np.random.default_rng(11)
    for sign, name in ((+1.0, "singlet"), (-1.0, "triplet")):
        E_exact = h[0, 0] + h[1, 1] + J12 + sign * K12
        coef = np.array([1.0, sign]) / np.sqrt(2.0)
        for _ in range(4):
            pa = rng.standard_normal((2, 1)) + 1j * rng.standard_normal((2, 1))
            pb = rng.standard_normal((2, 1)) + 1j * rng.standard_normal((2, 1))
            E = oracle.local_energy_cas_u([Cmo, Cmo], cols, coef, [Lbar, Lbar], [hbar, hbar], [fs, fs], [pa, pb])
            assert abs(E[0] - E_exact) <= 1e-12 * max(1.0, abs(E_exact)), (name, E[0], E_exact)
            assert abs(E[1] + E[2] + E[3] - E[0]) <= 1e-13


def test_pair_screening_bounds_and_energy_screen():
    """Pins of the oracle's pair screening on an extended geometry (24-site chain, where
    distant pairs really are negligible).  (i) The pre-SVD bounds form the chain sigma_1 <= |Y|_F <= sum_g |l^g_i||l^g_j| <=
    |Lbar_i|_F |Lbar_j|_F against LAPACK's sigma_1 of numpy-formed blocks, the triangle bound decays with |i-j| while the
    Cauchy-Schwarz one does not, and every pair whose bound is <= T has rank 0 in the oracle's own factor set.  (ii) The
    energy screen drops exactly the pairs with m_ij sigma_1 <= cutoff: the screened exchange plus the dropped pairs' own
    contributions (typed here with numpy from the full blocks) gives back the unscreened exchange, and the change stays
    inside sum_dropped m_ij sigma_1 |Theta_i||Theta_j|; cutoff 0 drops nothing, a huge cutoff everything."""
    xyz, fns = gen.chain_geometry(24, 3)
    P = gen.make_problem_from_geometry(xyz, fns, (24,), 120, seed=3)
    O, T = 24, 1e-5
    Lbar, hbar = oracle.half_rotate(P.L, P.h, P.psi[0])
    pi, pj = oracle.all_pairs(O)
    fro, tri, cs = oracle.pair_norm_bounds(Lbar, pi, pj)
    Ys = [Lbar[:, i, :].T @ Lbar[:, j, :] for i, j in zip(pi, pj)]
    s1 = np.array([np.linalg.svd(Y, compute_uv=False)[0] for Y in Ys])
    assert (s1 <= fro * (1 + 1e-12)).all() and (fro <= tri * (1 + 1e-12)).all() and (tri <= cs * (1 + 1e-12)).all()
    assert np.abs(fro - np.array([np.linalg.norm(Y) for Y in Ys])).max() <= 1e-12 * fro.max()
    far, near = (pj - pi) >= 16, (pj - pi) <= 1
    assert tri[far].max() < 1e-4 * tri[near].min() and cs[far].min() > 0.1 * cs[near].max()
    own = oracle.own_factors(Lbar, T)
    pre = tri <= T
    assert pre.sum() >= 20 and (own.r[pre] == 0).all() and (own.r[~pre] > 0).sum() >= 200
    # energy screen
    phis = gen.make_walkers(P, 3)
    full = oracle.own_factors(Lbar, 1e-9)
    fs0, drop0, ms1 = oracle.screen_pairs(full, 0.0)
    assert not drop0.any() and np.array_equal(fs0.r, full.r) and np.array_equal(fs0.U, full.U)
    m = np.where(pi == pj, 1.0, 2.0)
    assert np.abs(ms1 - m * s1).max() <= 1e-10 * s1.max()
    fs_inf, drop_inf, _ = oracle.screen_pairs(full, 1e30)
    assert fs_inf.sum_rank == 0 and drop_inf.sum() == (full.r > 0).sum()
    for cutoff in (1e-6, 1e-3, 0.3):
        fsc, drop, _ = oracle.screen_pairs(full, cutoff)
        assert np.array_equal(drop, (full.r > 0) & (m * s1 <= cutoff * (1 + 1e-12))) and 0 < drop.sum() < len(pi)
        for w in range(3):
            th, _, _ = oracle.theta(P.psi[0], phis[0][w])
            nrm = np.linalg.norm(th, axis=0)
            ek_full, ek_scr = oracle.exchange_lo(full, th), oracle.exchange_lo(fsc, th)
            dropped = sum(-m[k] * (th[:, pj[k]] @ Ys[k] @ th[:, pi[k]]) for k in np.nonzero(drop)[0])     # Eq. 17 per pair
            assert abs(ek_scr + dropped - ek_full) <= 1e-8 * abs(ek_full) + 1e-9 * (m * s1 * nrm[pi] * nrm[pj])[drop].sum() + 1e-12
            assert abs(ek_scr - ek_full) <= (m * s1 * nrm[pi] * nrm[pj])[drop].sum() * (1 + 1e-9)


def test_randomized_svd_pins():
    """Pins of oracle.randomized_svd (NEXT-4).  (i) A matrix of exact rank 9 built from known singular values
    and orthonormal factors: the sketch (k = 16) returns those singular values to 1e-12, a residual at rounding level and
    the same truncated matrix as LAPACK.  (ii) A full-rank block: the reported residual is the true error of the rank-k
    approximation, never below the optimum sqrt(sum_{K>k} sigma_K^2) (Eckart-Young) -- what lets a caller reject the
    sketch -- and every returned singular value is within resid of LAPACK's (Weyl).  (iii) A rank-deficient pair block
    of the "vector" reading of the generator."""
    rng = np.random.default_rng(5)
    n, r, k = 40, 9, 16
    A, _ = np.linalg.qr(rng.standard_normal((n, n)))
    Bm, _ = np.linalg.qr(rng.standard_normal((n, n)))
    sig = np.array([7.0, 3.0, 2.5, 1.0, 0.3, 0.1, 1e-2, 1e-4, 1e-6])
    Y = (A[:, :r] * sig) @ Bm[:, :r].T
    Ut, s, Wt, resid = oracle.randomized_svd(Y, rng.standard_normal((n, k)))
    assert np.abs(s[:r] - sig).max() <= 1e-12 * sig[0] and s[r:].max() <= 1e-13 * sig[0] and resid <= 1e-13 * sig[0]
    assert np.abs((Ut[:r].T * s[:r]) @ Wt[:r] - Y).max() <= 1e-13 * sig[0]
    assert np.abs(np.abs(np.sum(Ut[:r] * A[:, :r].T, axis=1)) - 1).max() <= 1e-9        # same vectors up to sign
    assert np.abs(Ut @ Ut.T - np.eye(k)).max() <= 1e-12 and np.abs(Wt @ Wt.T - np.eye(k)).max() <= 1e-12
    Yf = rng.standard_normal((n, n)) * np.exp(-0.2 * np.arange(n))[None, :]
    sl = np.linalg.svd(Yf, compute_uv=False)
    Ut, s, Wt, resid = oracle.randomized_svd(Yf, rng.standard_normal((n, k)))
    assert resid >= np.sqrt((sl[k:] ** 2).sum()) * (1 - 1e-12) and resid <= 20 * np.sqrt((sl[k:] ** 2).sum())
    assert np.abs(np.linalg.norm(Yf - (Ut.T * s) @ Wt) - resid) <= 1e-12 * sl[0]
    assert (np.abs(s - sl[:k]) <= resid * (1 + 1e-12)).all()
    P = gen.make_problem(0, reading="vector")
    Lbar, _ = oracle.half_rotate(P.L, P.h, P.psi[0])
    Yv = oracle.pair_eri(Lbar, 1, 4)
    slv = np.linalg.svd(Yv, compute_uv=False)
    assert (slv > 1e-10 * slv[0]).sum() <= 4                                       # rank <= number of sites
    Ut, s, Wt, resid = oracle.randomized_svd(Yv, rng.standard_normal((P.N, 8)))
    assert resid <= 1e-13 * slv[0] and np.abs(s[:4] - slv[:4]).max() <= 1e-12 * slv[0]
