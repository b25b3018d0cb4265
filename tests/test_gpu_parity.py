"""GPU parity tests (run with -m gpu on the B200 box): the CUDA path, called through the C ABI, against the CPU oracle
on the same seeded inputs and -- protocol (A) of SURVEY.md 8(c) -- on the LIBRARY's factor set.
Tolerance (BASELINE.json:north_star): |dE|/|E_L| <= 1e-10 per walker, for E_L and for every part."""
import numpy as np
import pytest

import gen
import oracle
import paper_2202_00832_b200 as lo

pytestmark = pytest.mark.gpu
TOL = 1e-10


def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")
    return torch


def oracle_factor_sets(P, F):
    fs = []
    for s in range(P.n_spin):
        U, sg, W = F.factor_all(s)
        pi, pj = oracle.all_pairs(P.n_occ[s])
        fs.append(oracle.make_factor_set(P.N, P.n_occ[s], pi, pj, F.ranks(s), U, sg, W))
    return fs


def oracle_energy(P, F, phis, idx=None):
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]
    sel = [p if idx is None else p[idx] for p in phis]
    return oracle.local_energy_lo(P.psi, [a for a, _ in hr], [b for _, b in hr], oracle_factor_sets(P, F), sel)


def oracle_energy_streamed(P, F, phis, idx, chunk=128):
    """Protocol (A) for factor sets too large to copy to the host in one piece: the oracle's exchange sum is
    accumulated over chunks of pairs fetched from the library (lo_factor_pair)."""
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]

    def fetch(spin, k0, k1):
        r, U, sg, W = F.factor_range(spin, k0, k1)
        pi, pj = oracle.all_pairs(P.n_occ[spin])
        return oracle.make_factor_set(P.N, P.n_occ[spin], pi[k0:k1], pj[k0:k1], r, U, sg, W)

    n_pairs = [o * (o + 1) // 2 for o in P.n_occ]
    E, st, _ = oracle.local_energy_lo_streamed(P.psi, [a for a, _ in hr], [b for _, b in hr], [p[idx] for p in phis], n_pairs, fetch, chunk)
    return E, st


def gpu_energy(F, phis):
    torch = torch_cuda()
    d = [torch.from_numpy(np.ascontiguousarray(p)).cuda() for p in phis]
    out = F.local_energy(d)
    torch.cuda.synchronize()
    E = np.stack([e.cpu().numpy() for e in out[:4]], axis=1)
    return E, out[4].cpu().numpy()


def assert_parity(Eg, Eo, tol=TOL):
    scale = np.abs(Eo[:, 0:1])
    err = np.abs(Eg - Eo) / scale
    assert err.max() <= tol, "max rel err per part (E_L,E1,E_J,E_K) = %s" % err.max(axis=0)
    assert np.abs(Eg[:, 0] - Eg[:, 1:].sum(axis=1)).max() <= 1e-12 * np.abs(Eg).max()


def assert_close(Ea, Eb, what, tol=1e-12):
    """Two launch configurations of the same arithmetic (different fixed summation orders): 1e-12 of |E_L| per walker."""
    err = np.abs(Ea - Eb).max(axis=1) / np.abs(Eb[:, 0])
    assert err.max() <= tol, "%s differs: max rel %.2e on walker %d" % (what, err.max(), int(err.argmax()))
    return True


def assert_all_walkers(P, F, phis, Eg, stride=1):
    """Properties that hold at any size, on walkers the sampled oracle check does not visit: (i) repeated calls are
    bitwise equal on EVERY walker and every part (fixed-order reductions; this is what exposes a pipeline race) and the
    host-buffer variant agrees to 1e-12 of |E_L| (it runs the batch in walker chunks: the same arithmetic per walker in
    another fixed summation order of the partials), (ii) E1 and E_J of every stride-th walker against the oracle (Theta,
    one-body, Cholesky Coulomb: cheap enough for whole batches), E_L = E1 + E_J + E_K on all."""
    torch = torch_cuda()
    for _ in range(2):
        E2, _ = gpu_energy(F, phis)
        assert np.array_equal(E2, Eg), "repeated call differs on walkers %s" % np.nonzero((E2 != Eg).any(axis=1))[0][:8]
    Eh, sh = F.local_energy_host([torch.from_numpy(np.ascontiguousarray(p)).pin_memory() for p in phis])
    # the host variant runs the batch in walker chunks (copy/compute overlap): same arithmetic per walker, but the
    # fixed summation order of the split-K / per-CTA partials depends on the number of walker blocks in a launch
    assert_close(Eh, Eg, "host-buffer variant")
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]
    empty = [oracle.empty_factor_set(P.N, o) for o in P.n_occ]
    sel = [p[::stride] for p in phis]
    Eo, _ = oracle.local_energy_lo(P.psi, [a for a, _ in hr], [b for _, b in hr], empty, sel)
    scale = np.abs(Eg[::stride, 0:1])
    err = np.abs(Eg[::stride, 1:3] - Eo[:, 1:3]) / scale
    assert err.max() <= TOL, "E1/E_J of all walkers: max rel err %s at walker %d" % (err.max(axis=0), stride * int(err.max(axis=1).argmax()))


# ------------------------------------------------------------------------------------------ C0, C1: every walker
@pytest.mark.parametrize("gpu_svd", [False, True])
def test_c0_all_walkers(c0, gpu_svd):
    phis = gen.make_walkers(c0)
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=0, max_walkers=c0.n_w, gpu_svd=gpu_svd)
    Eg, st = gpu_energy(F, phis)
    Eo, so = oracle_energy(c0, F, phis)
    assert (st == 0).all() and (so == 0).all()
    assert_parity(Eg, Eo)
    # untruncated in effect (T=1e-8 keeps all 24 values): equals the exact brute-force energy (Eq. 10) as well
    for w in range(c0.n_w):
        e = np.array(oracle.local_energy_exact(c0.h, c0.L, c0.psi, [phis[0][w]], "bruteforce"))
        assert np.abs(Eg[w] - e).max() <= 1e-9 * abs(e[0])


@pytest.mark.parametrize("T", [1e-4, 1e-6])
def test_c1_all_walkers(c1, T):
    phis = gen.make_walkers(c1)
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, T, device=0, max_walkers=c1.n_w, gpu_svd=True)
    Eg, st = gpu_energy(F, phis)
    Eo, _ = oracle_energy(c1, F, phis)
    assert (st == 0).all()
    assert_parity(Eg, Eo)


def test_c1_theta_parity(c1):
    phis = gen.make_walkers(c1, 40)
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1.0, device=0, max_walkers=40)
    gpu_energy(F, phis)
    th = F.theta_host(0, 40)
    for w in range(40):
        tho, _, _ = oracle.theta(c1.psi[0], phis[0][w])
        assert np.abs(th[w] - tho).max() <= 1e-12 * np.abs(tho).max()
        assert np.abs(c1.psi[0].T @ th[w] - np.eye(c1.n_occ[0])).max() < 1e-11      # Psi^T Theta = I


# ------------------------------------------------------------------------------------------ small / ragged ranks
def test_c1_vector_reading_small_ragged_ranks():
    P = gen.make_problem(1, reading="vector")
    phis = gen.make_walkers(P, 100)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-4, device=0, max_walkers=128, gpu_svd=True)
    r = F.ranks()
    assert r.max() <= 12 and r.min() < r.max()
    Eg, _ = gpu_energy(F, phis)
    Eo, _ = oracle_energy(P, F, phis)
    assert_parity(Eg, Eo)
    # a looser threshold through lo_retruncate: ragged ranks incl. zeros, still parity on that factor set
    F2 = F.retruncate(0.05)
    r2 = F2.ranks()
    assert r2.sum() < r.sum()
    Eg2, _ = gpu_energy(F2, phis)
    Eo2, _ = oracle_energy(P, F2, phis)
    assert_parity(Eg2, Eo2)


@pytest.mark.parametrize("n_w", [1, 5, 17, 33, 48, 49, 64, 65, 130])
def test_ragged_walker_counts(c1, n_w):
    phis = gen.make_walkers(c1, n_w, seed=99)
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 5.0, device=0, max_walkers=130)
    Eg, st = gpu_energy(F, phis)
    Eo, _ = oracle_energy(c1, F, phis)
    assert Eg.shape == (n_w, 4)
    assert_parity(Eg, Eo)


def test_all_pairs_truncated_away(c0):
    phis = gen.make_walkers(c0)
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e9, device=0, max_walkers=8)
    assert F.info().sum_rank[0] == 0
    Eg, _ = gpu_energy(F, phis)
    assert (Eg[:, 3] == 0).all()
    Eo, _ = oracle_energy(c0, F, phis)
    assert_parity(Eg, Eo)


# ------------------------------------------------------------------------------------------ unrestricted (O6)
def test_unrestricted_small():
    xyz, fns = gen.site_geometry(1)
    P = gen.make_problem_from_geometry(xyz, fns, (9, 7), 300, seed=31)
    phis = gen.make_walkers(P, 70)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-6, device=0, max_walkers=70, gpu_svd=True)
    Eg, st = gpu_energy(F, phis)
    Eo, _ = oracle_energy(P, F, phis)
    assert_parity(Eg, Eo)
    for w in (0, 33):
        e = np.array(oracle.local_energy_exact(P.h, P.L, P.psi, [phis[0][w], phis[1][w]], "cholesky"))
        assert np.abs(Eg[w] - e).max() <= 1e-4 * abs(e[0])      # T=1e-6: close to exact
    # identical alpha/beta inputs reproduce the closed-shell result (P9)
    P2 = gen.make_problem_from_geometry(xyz, fns, (9,), 300, seed=31)
    Fr = lo.Factors.setup(P2.h, P2.L, P2.psi, 1e-6, device=0, max_walkers=70)
    Fu = lo.Factors.setup(P2.h, P2.L, [P2.psi[0], P2.psi[0]], 1e-6, device=0, max_walkers=70)
    ph = gen.make_walkers(P2, 70)
    Er, _ = gpu_energy(Fr, ph)
    Eu, _ = gpu_energy(Fu, [ph[0], ph[0]])
    assert np.abs(Er - Eu).max() <= 1e-12 * np.abs(Er).max()


# ------------------------------------------------------------------------------------------ degenerate inputs
def test_singular_walker_is_flagged(c0):
    phis = gen.make_walkers(c0)
    phi = phis[0].copy()
    phi[3, :, 1] = 0.0                          # a zero orbital: exactly singular overlap (zero pivot on both sides)
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=0, max_walkers=8)
    Eg, st = gpu_energy(F, [phi])
    Eo, so = oracle_energy(c0, F, [phi])
    assert st[3] == 1 and so[3] == 1 and st.sum() == 1
    assert np.isnan(Eg[3]).all() and np.isnan(Eo[3]).all()
    ok = [w for w in range(8) if w != 3]
    assert_parity(Eg[ok], Eo[ok])


def test_trial_walker_gives_hf_energy(c1):
    psi = c1.psi[0]
    D = psi @ psi.T
    LD = np.einsum("gpq,qr->gpr", c1.L, D)
    e_hf = 2 * np.trace(c1.h @ D) + 2 * (np.trace(LD, axis1=1, axis2=2) ** 2).sum() - np.einsum("gpr,grp->", LD, LD)
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 0.0, device=0, max_walkers=2, gpu_svd=True)
    Eg, st = gpu_energy(F, [np.stack([psi, psi]).astype(np.complex128)])
    assert abs(Eg[0, 0].real - e_hf) <= 1e-10 * abs(e_hf) and abs(Eg[0, 0].imag) <= 1e-10 * abs(e_hf)


# ------------------------------------------------------------------------------------------ API variants
def test_host_variant_and_determinism(c1):
    torch = torch_cuda()
    phis = gen.make_walkers(c1, 300)    # host variant: 2 walker chunks (64 + a ragged 236)
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=300, gpu_svd=True)
    E1, _ = gpu_energy(F, phis)
    E2, _ = gpu_energy(F, phis)
    assert np.array_equal(E1, E2)                                  # fixed-order reductions: bitwise repeatable
    pinned = [torch.from_numpy(p).pin_memory() for p in phis]
    Eh, sh = F.local_energy_host(pinned)
    assert_close(Eh, E1, "host-buffer variant") and (sh == 0).all()
    Eh2, _ = F.local_energy_host(phis)                              # pageable numpy buffers
    assert np.array_equal(Eh2, Eh)                                  # the host variant is bitwise repeatable too
    assert_close(Eh2, E1, "host-buffer variant (pageable)")
    e_only = F.local_energy([torch.from_numpy(p).cuda() for p in phis], parts=False, status=False)
    torch.cuda.synchronize()
    assert np.array_equal(e_only[0].cpu().numpy(), E1[:, 0])
    with pytest.raises(lo.LoError):
        F.local_energy([torch.from_numpy(gen.make_walkers(c1, 301)[0]).cuda()])     # n_w > max_walkers


def test_gpu_svd_matches_host_svd(c1):
    Fh = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=8, gpu_svd=False)
    Fg = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=8, gpu_svd=True)
    assert np.array_equal(Fh.ranks(), Fg.ranks())
    assert Fg.info().setup_on_gpu == 1 and Fh.info().setup_on_gpu == 0
    for (i, j) in [(0, 0), (4, 11), (20, 20)]:
        Uh, sh, Wh = Fh.factor_pair(0, i, j)
        Ug, sg, Wg = Fg.factor_pair(0, i, j)
        assert np.abs(sh - sg).max() <= 1e-12 * sh[0]
        assert np.abs((Uh.T * sh) @ Wh - (Ug.T * sg) @ Wg).max() <= 1e-11 * sh[0]
        assert np.abs(Ug @ Ug.T - np.eye(len(sg))).max() < 1e-12
    # protocol (B): oracle on its own factors vs oracle on the library's factors
    phis = gen.make_walkers(c1, 4)
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, c1.psi[0])
    own = oracle.own_factors(Lbar, 1e-4)
    assert np.array_equal(own.r, Fg.ranks())
    E_own, _ = oracle.local_energy_lo(c1.psi, [Lbar], [hbar], [own], phis)
    E_lib, _ = oracle_energy(c1, Fg, phis)
    assert np.abs(E_own - E_lib).max() <= 1e-9 * np.abs(E_own[:, 0]).min()


def test_gpu_factors_pinned_to_lapack(c1, c2_built):
    """The device setup path (LO_SETUP_GPU_SVD: k_pair_gram + the block Jacobi of lo_svd.cu) against LAPACK
    (numpy.linalg.svd of Y^{ij} formed by numpy -- no SVD routine of this repo, oracle or product, takes part): all 231 pair
    blocks of configs[1] and 64 |i-j|-stratified pair blocks of configs[2] (378 x 378): singular values to 1e-12 sigma_1,
    rank vectors equal outside the band |sigma - T| <= 1e-10 sigma_max (DESIGN R13), truncated reconstructions to
    1e-11 sigma_1, orthonormal factor rows.  This is what makes the library's factors independent of the oracle's SVD."""
    from test_abi_host import lapack_pin
    O = c1.n_occ[0]
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=8, gpu_svd=True)
    info = F.info()
    assert info.setup_on_gpu == 1 and 2 <= info.svd_sweeps_max < 40 and info.svd_offdiag_max <= c1.N * 2.0 ** -53
    Lbar = np.einsum("gpq,qi->gip", c1.L, c1.psi[0])
    assert lapack_pin(F, 0, Lbar, [(i, j) for i in range(O) for j in range(i, O)], 1e-4, c1.N) <= 2
    P, _, F2 = c2_built
    O2 = P.n_occ[0]
    Lbar2 = np.einsum("gpq,qi->gip", P.L, P.psi[0])
    pi, pj = np.triu_indices(O2)
    order = np.argsort(pj - pi, kind="stable")
    sel = order[np.linspace(0, len(pi) - 1, 64).astype(int)]
    assert lapack_pin(F2, 0, Lbar2, [(int(pi[k]), int(pj[k])) for k in sel], 1e-5, P.N) <= 2
    i2 = F2.info()
    assert 2 <= i2.svd_sweeps_max < 40 and i2.svd_offdiag_max <= P.N * 2.0 ** -53


def test_randomized_svd_setup_device_path(c1):
    """LO_SETUP_RANDOMIZED_SVD on the device.  configs[2] in the rank-deficient "vector"
    reading (ranks 23..36, sketch of 64 rows): every pair block is accepted by the a-posteriori check, the factors pass the
    LAPACK pin (32 |i-j|-stratified pairs) and give the same ranks as the full method, and the energies of 8 walkers match
    the oracle on that factor set (1e-10).  configs[1] in the full-rank reading: every sketch is rejected and the factor set is
    the full method's bit for bit."""
    from test_abi_host import lapack_pin
    P = gen.make_problem(2, reading="vector")
    Fr = lo.Factors.setup(P.h, P.L, P.psi, 1e-5, device=0, max_walkers=8, gpu_svd=True, rsvd=64)
    Ff = lo.Factors.setup(P.h, P.L, P.psi, 1e-5, device=0, max_walkers=8, gpu_svd=True)
    ir, iff = Fr.info(), Ff.info()
    assert ir.rsvd_sketch == 64 and ir.n_pairs_rsvd == ir.n_pairs[0] and iff.n_pairs_rsvd == 0
    assert np.array_equal(Fr.ranks(), Ff.ranks()) and Fr.ranks().max() <= 36
    print("setup seconds (SVD part): randomised %.2f (%.2f), full %.2f (%.2f)" % (ir.setup_seconds, ir.setup_svd_seconds, iff.setup_seconds, iff.setup_svd_seconds))
    Lbar = np.einsum("gpq,qi->gip", P.L, P.psi[0])
    pi, pj = np.triu_indices(P.n_occ[0])
    order = np.argsort(pj - pi, kind="stable")
    sel = order[np.linspace(0, len(pi) - 1, 32).astype(int)]
    lapack_pin(Fr, 0, Lbar, [(int(pi[k]), int(pj[k])) for k in sel], 1e-5, P.N)
    phis = gen.make_walkers(P, 8)
    Eg, st = gpu_energy(Fr, phis)
    Eo, _ = oracle_energy(P, Fr, phis)
    assert (st == 0).all()
    assert_parity(Eg, Eo)
    Fe = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=8, gpu_svd=True, rsvd=16)
    Fe0 = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=8, gpu_svd=True)
    assert Fe.info().n_pairs_rsvd == 0
    for a, b in zip(Fe.factor_all(), Fe0.factor_all()):
        assert np.array_equal(a, b)


def test_exact_energy_within_truncation_bound():
    # protocol (C): GPU LO energy vs the exact exchange, inside the bound of SURVEY 8c-D14
    P = gen.make_problem(1, reading="vector")
    phis = gen.make_walkers(P, 8)
    Lbar, hbar = oracle.half_rotate(P.L, P.h, P.psi[0])
    pi, pj = oracle.all_pairs(P.n_occ[0])
    m = np.where(pi == pj, 1.0, 2.0)
    for T in (1e-4, 0.05, 0.5):
        F = lo.Factors.setup(P.h, P.L, P.psi, T, device=0, max_walkers=8, gpu_svd=True)
        Eg, _ = gpu_energy(F, phis)
        for w in range(8):
            th, _, _ = oracle.theta(P.psi[0], phis[0][w])
            nrm = np.linalg.norm(th, axis=0)
            ek = oracle.exchange_cholesky(Lbar, th)
            assert abs(Eg[w, 3] - ek) <= T * (m * nrm[pi] * nrm[pj]).sum() + 1e-10 * abs(ek)


def test_coulomb_x_export(c1):
    import ctypes
    torch = torch_cuda()
    phis = gen.make_walkers(c1, 10)
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 5.0, device=0, max_walkers=10)
    gpu_energy(F, phis)
    ptr, ld = F.coulomb_x()
    X = np.empty((c1.n_chol, ld), dtype=np.complex128)
    cudart = ctypes.CDLL("libcudart.so")
    assert cudart.cudaMemcpy(ctypes.c_void_p(X.ctypes.data), ctypes.c_void_p(ptr), ctypes.c_size_t(X.nbytes), 2) == 0
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, c1.psi[0])
    for w in (0, 9):
        th, _, _ = oracle.theta(c1.psi[0], phis[0][w])
        _, _, Xo = oracle.onebody_coulomb([Lbar], [hbar], [th], want_X=True)
        assert np.abs(X[:, w] - Xo).max() <= 1e-12 * np.abs(Xo).max()


# ------------------------------------------------------------------------------------------ full size, sampled outputs
@pytest.fixture(scope="module")
def c2_built():
    """configs[2] factor set (T = 1e-5, device setup), built once for the tests that use it."""
    P = gen.make_problem(2)
    phis = gen.make_walkers(P)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-5, device=0, max_walkers=P.n_w, gpu_svd=True)
    yield P, phis, F
    F.free()


def test_c2_full_size_sampled_walkers(c2_built):
    """BASELINE.json:configs[2] (pentacene-sized, headline) in bench.py's launch configuration: all 512 walkers on
    the GPU; 64 seeded walkers checked one by one by the oracle on the library's factor set (a seeded subset
    of >= 64 walkers); E1/E_J of every walker, repeatability and the host-buffer variant on all walkers."""
    P, phis, F = c2_built
    info = F.info()
    assert info.n_pairs[0] == 73 * 74 // 2 and info.max_rank <= 378
    Eg, st = gpu_energy(F, phis)
    assert (st == 0).all() and np.isfinite(Eg).all()
    idx = np.random.default_rng(2).choice(P.n_w, 64, replace=False)
    Eo, _ = oracle_energy(P, F, phis, idx)
    assert_parity(Eg[idx], Eo)
    assert_all_walkers(P, F, phis, Eg)
    # exact Cholesky-route exchange for two walkers: inside the truncation bound
    Lbar, _ = oracle.half_rotate(P.L, P.h, P.psi[0])
    pi, pj = oracle.all_pairs(73)
    m = np.where(pi == pj, 1.0, 2.0)
    for w in idx[:2]:
        th, _, _ = oracle.theta(P.psi[0], phis[0][w])
        nrm = np.linalg.norm(th, axis=0)
        ek = oracle.exchange_cholesky(Lbar, th)
        assert abs(Eg[w, 3] - ek) <= 1e-5 * (m * nrm[pi] * nrm[pj]).sum() + 1e-10 * abs(ek)


def test_c3_full_size_unrestricted_sampled_walkers():
    """BASELINE.json:configs[3] (open-shell metallocene-sized, N=500, 65 alpha + 63 beta, N_chol=2500, T=1e-5): all
    1024 walkers on the GPU, 64 seeded walkers (>= 64) checked one by one by the oracle on the library's
    factor set (exchange streamed in chunks of pairs: the 2 x 8 GB of factors do not need to sit on the host at once)."""
    P = gen.make_problem(3)
    phis = gen.make_walkers(P)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-5, device=0, max_walkers=P.n_w, gpu_svd=True)
    info = F.info()
    assert tuple(info.n_pairs) == (65 * 66 // 2, 63 * 64 // 2) and info.n_spin == 2
    Eg, st = gpu_energy(F, phis)
    assert (st == 0).all() and np.isfinite(Eg).all()
    idx = np.sort(np.random.default_rng(3).choice(P.n_w, 64, replace=False))
    Eo, so = oracle_energy_streamed(P, F, phis, idx)
    assert (so == 0).all()
    assert_parity(Eg[idx], Eo)
    assert_all_walkers(P, F, phis, Eg)
    # the same batch on the INT8 route (exchange of both spins and the Coulomb term summed over both spins from digit slices):
    # the sampled walkers against the oracle, every walker against the DMMA route
    Eq, sq = int8_energy(F, phis)
    assert (sq == 0).all()
    assert_parity(Eq[idx], Eo)
    assert_close(Eq, Eg, "INT8 route vs DMMA route, configs[3]", tol=1e-10)


def test_c4_threshold_sweep_parity():
    """BASELINE.json:configs[4] (3D cage, N=700, N_occ=130, N_chol=3500, 2048 walkers, thresholds 1e-3 .. 1e-6): the
    factor set is built ONCE at T = 1e-6 (the pair SVDs are full whatever T is; 67 GB of factors, 64-bit row offsets) and
    re-truncated to 1e-5, 1e-4, 1e-3 (lo_retruncate, prefix truncation).  At EACH threshold all 2048 walkers run on the
    GPU in bench.py's launch configuration and a seeded subset is checked one by one by the oracle on that factor set
    (protocol A, 1e-10 per walker and part; exchange streamed in chunks of pairs): 32 walkers at 1e-6, 8 walkers at each
    of the other three; E1/E_J of every 4th walker, repeatability and the host-buffer variant on all walkers at 1e-6."""
    P = gen.make_problem(4)
    phis = gen.make_walkers(P)
    F6 = lo.Factors.setup(P.h, P.L, P.psi, 1e-6, device=0, max_walkers=P.n_w, gpu_svd=True)
    info = F6.info()
    assert info.n_pairs[0] == 130 * 131 // 2 and info.max_rank <= 700 and info.factor_bytes > 60e9
    assert info.svd_sweeps_max < 40 and info.svd_offdiag_max <= 700 * 2.0 ** -53
    idx = np.sort(np.random.default_rng(4).choice(P.n_w, 32, replace=False))
    sums = []
    for T, n_chk in [(1e-6, 32), (1e-5, 8), (1e-4, 8), (1e-3, 8)]:
        F = F6 if T == 1e-6 else F6.retruncate(T)
        assert F.info().threshold == T
        sums.append(int(F.info().sum_rank[0]))
        Eg, st = gpu_energy(F, phis)
        assert (st == 0).all() and np.isfinite(Eg).all()
        Eo, so = oracle_energy_streamed(P, F, phis, idx[:n_chk])
        assert (so == 0).all()
        assert_parity(Eg[idx[:n_chk]], Eo)
        if F is F6:
            assert_all_walkers(P, F, phis, Eg, stride=4)
        else:
            F.free()
    assert sums[0] > sums[1] > sums[2] > sums[3] > 0          # sum r_ij falls with the threshold (P8)
    F6.free()


def exchange_tile_fragments(ranks):
    """Fragment counts (8-row fragments, 1..8) of the row tiles lo_setup cuts for these ranks: ceil(r/8) fragments in
    ceil(fragments/8) tiles of near-equal size (include/lo_afqmc.h, lo_info.n_tiles)."""
    out = []
    for r in ranks:
        f8 = (int(r) + 7) // 8
        nt = (f8 + 7) // 8
        out += [f8 // nt + (1 if t < f8 % nt else 0) for t in range(nt)]
    return out


@pytest.mark.parametrize("n_w", [64, 65, 16])
def test_every_tile_fragment_count(c1, n_w):
    """A factor set whose row tiles take EVERY fragment count 1..8 (configs[1] re-truncated at T = 3, a value inside its
    own singular-value spectrum: ranks 1..82), so that each instantiation ex_kloop<1..8> of the exchange kernels runs; parity
    per walker and part at a full block (64 walkers), a ragged batch (65) and the narrow-batch kernel (16)."""
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=n_w, gpu_svd=True).retruncate(3.0)
    frags = exchange_tile_fragments(F.ranks())
    assert set(frags) == set(range(1, 9)) and len(frags) == F.info().n_tiles
    phis = gen.make_walkers(c1, n_w, seed=7)
    Eg, st = gpu_energy(F, phis)
    Eo, _ = oracle_energy(c1, F, phis)
    assert (st == 0).all()
    assert_parity(Eg, Eo)
    F.set_coulomb_mode(True)                                   # NEXT-3 kernel instantiation (tiles of <= 4 fragments)
    Eg2, _ = gpu_energy(F, phis)
    fs = oracle_factor_sets(c1, F)[0]
    for w in (0, n_w - 1):
        th, _, _ = oracle.theta(c1.psi[0], phis[0][w])
        assert abs(Eg2[w, 2] - 2.0 * oracle.coulomb_lo(fs, th)) <= TOL * abs(Eo[w, 0])      # closed shell: E_J^LO = 2 S
        assert abs(Eg2[w, 3] - Eo[w, 3]) <= TOL * abs(Eo[w, 0])


# ------------------------------------------------------------------------------------------ NEXT-4: pair screening
def test_pair_screening_on_a_chain():
    """SURVEY 8(f) NEXT-4 / PAPER.md:318 on an extended geometry (40-site chain, N = 120, 820 pairs), device setup path.
    (i) Rigorous pre-SVD screen: with and without it the factor set is bit-identical (ranks, rows, singular values, tiles),
    lo_info counts the pairs that were never decomposed.  (ii) Energy screen (lo_screen_pairs): GPU parity with the oracle
    on the screened factor set (1e-10), the same pairs dropped as by the oracle's plain-loop rule, and the change of E_K of
    every walker inside  sum_dropped m_ij sigma_1 |Theta_i||Theta_j|."""
    xyz, fns = gen.chain_geometry(40, 3)
    P = gen.make_problem_from_geometry(xyz, fns, (40,), 600, seed=3)
    T, n_w = 1e-6, 70
    Fs = lo.Factors.setup(P.h, P.L, P.psi, T, device=0, max_walkers=n_w, gpu_svd=True)
    Fn = lo.Factors.setup(P.h, P.L, P.psi, T, device=0, max_walkers=n_w, gpu_svd=True, prescreen=False)
    i_s, i_n = Fs.info(), Fn.info()
    assert i_n.n_pairs_prescreened == 0 and i_s.n_pairs_prescreened > 100
    assert np.array_equal(Fs.ranks(), Fn.ranks()) and i_s.n_tiles == i_n.n_tiles
    for a, b in zip(Fs.factor_all(), Fn.factor_all()):
        assert np.array_equal(a, b)
    assert (Fs.ranks() == 0).sum() >= i_s.n_pairs_prescreened
    phis = gen.make_walkers(P, n_w)
    E0, _ = gpu_energy(Fs, phis)
    assert np.array_equal(E0, gpu_energy(Fn, phis)[0])
    assert_parity(E0, oracle_energy(P, Fs, phis)[0])
    pi, pj = oracle.all_pairs(40)
    fs = oracle_factor_sets(P, Fs)[0]
    m = np.where(pi == pj, 1.0, 2.0)
    kept = []
    for cutoff in (1e-4, 1e-2):
        Fc = Fs.screen_pairs(cutoff)
        fso, drop, ms1 = oracle.screen_pairs(fs, cutoff)
        assert np.array_equal(Fc.ranks(), fso.r) and Fc.info().n_pairs_energy_screened == int(drop.sum()) > 0
        Ec, st = gpu_energy(Fc, phis)
        Eo, _ = oracle_energy(P, Fc, phis)
        assert (st == 0).all()
        assert_parity(Ec, Eo)
        for w in range(0, n_w, 7):
            th, _, _ = oracle.theta(P.psi[0], phis[0][w])
            nrm = np.linalg.norm(th, axis=0)
            assert abs(Ec[w, 3] - E0[w, 3]) <= (ms1 * nrm[pi] * nrm[pj])[drop].sum() * (1 + 1e-9)
            assert abs(Ec[w, 3] - E0[w, 3]) <= Fc.info().energy_screen_bound * nrm.max() ** 2 * (1 + 1e-9)
        kept.append(int((Fc.ranks() > 0).sum()))
    assert kept[1] < kept[0] < (Fs.ranks() > 0).sum() <= 820


# ------------------------------------------------------------------------------------------ NEXT-1: propagator
@pytest.mark.parametrize("n_w", [5, 130])
def test_propagator_matches_oracle(c1, n_w):
    """lo_propagator: B_w = sum_g x^g_w L^g for every walker of a ragged batch, element by element
    against the oracle's plain triple loop; 1e-13 of max|B_w| (a length-570 fp64 dot product in another order)."""
    torch = torch_cuda()
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=n_w, gpu_svd=True, propagator=True)
    rng = np.random.default_rng(11)
    x = rng.standard_normal((n_w, c1.n_chol)) + 1j * rng.standard_normal((n_w, c1.n_chol))
    F.propagator(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    ptr, ld, n_rows = F.propagator_buffer()
    assert n_rows == c1.N * (c1.N + 1) // 2 and ld >= n_w and ptr
    for w in ([0, 3, 4] if n_w == 5 else [0, 63, 64, 129]):
        Bo = oracle.propagator(c1.L, x[w])
        Bg = F.propagator_host(w)
        assert np.abs(Bg - Bo).max() <= 1e-13 * np.abs(Bo).max()
    # the energy path is untouched by the propagator call and its workspace
    phis = gen.make_walkers(c1, n_w)
    Eg, st = gpu_energy(F, phis)
    Eo, _ = oracle_energy(c1, F, phis)
    assert_parity(Eg, Eo)


def test_propagator_needs_flag(c0):
    torch = torch_cuda()
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=0, max_walkers=4, gpu_svd=True)
    with pytest.raises(lo.LoError):
        F.propagator(torch.zeros((4, c0.n_chol), dtype=torch.complex128, device="cuda"))


# ------------------------------------------------------------------------------------------ NEXT-3: compressed Coulomb
@pytest.mark.parametrize("T,reading", [(1e-4, "element"), (1e-2, "element"), (1e-6, "vector")])
def test_compressed_coulomb_mode(T, reading):
    """lo_set_coulomb_mode(COMPRESSED): E_J = 2 sum_{i<=j} m_ij sum_K sigma_K (U^T Theta_i)_K (W Theta_j)_K (Eq. 19/22
    first term) from the same tiles as the exchange, against the oracle's paper-literal sum on
    the library's factor set; E1 and E_K are those of the default mode bit for bit up to the tile cut (1e-10), and
    E_L = E1 + E_J^LO + E_K.  Ragged ranks (T=1e-2 truncates; the vector reading has ranks 11-12) and a ragged batch."""
    P = gen.make_problem(1, reading=reading)
    n_w = 70
    phis = gen.make_walkers(P, n_w)
    F = lo.Factors.setup(P.h, P.L, P.psi, T, device=0, max_walkers=n_w, gpu_svd=True)
    E_ch, _ = gpu_energy(F, phis)
    F.set_coulomb_mode(True)
    E_lo, st = gpu_energy(F, phis)
    assert (st == 0).all()
    fs = oracle_factor_sets(P, F)[0]
    scale = np.abs(E_ch[:, 0])
    for w in range(n_w):
        th, _, _ = oracle.theta(P.psi[0], phis[0][w])
        ej = 2.0 * oracle.coulomb_lo(fs, th)
        assert abs(E_lo[w, 2] - ej) <= TOL * scale[w]
    assert (np.abs(E_lo[:, 1] - E_ch[:, 1]) <= TOL * scale).all() and (np.abs(E_lo[:, 3] - E_ch[:, 3]) <= TOL * scale).all()
    assert (np.abs(E_lo[:, 0] - (E_lo[:, 1] + E_lo[:, 2] + E_lo[:, 3])) <= TOL * scale).all()
    # the compressed Coulomb term carries a truncation error of the same order as the exchange's
    if T >= 1e-2:
        assert np.abs(E_lo[:, 2] - E_ch[:, 2]).max() > 1e-9 * scale.max()
    # the same mode on the INT8 route (four projections per pair from the digit slices): every part against the DMMA result
    # and E_J against the oracle's paper-literal sum
    Eq, sq = int8_energy(F, phis)
    assert (sq == 0).all()
    assert_close(Eq, E_lo, "compressed Coulomb mode, INT8 route vs DMMA route", tol=1e-10)
    for w in (0, 33, 69):
        th, _, _ = oracle.theta(P.psi[0], phis[0][w])
        assert abs(Eq[w, 2] - 2.0 * oracle.coulomb_lo(fs, th)) <= TOL * scale[w]
    E_lo2, _ = gpu_energy(F, phis)
    assert np.array_equal(E_lo2, E_lo)
    F.set_coulomb_mode(False)
    E_back, _ = gpu_energy(F, phis)
    assert np.array_equal(E_back, E_ch)


def test_compressed_coulomb_exact_at_zero_threshold(c0, c0_walkers):
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 0.0, device=0, max_walkers=c0.n_w, gpu_svd=True)
    E_ch, _ = gpu_energy(F, c0_walkers)
    F.set_coulomb_mode(True)
    E_lo, _ = gpu_energy(F, c0_walkers)
    assert (np.abs(E_lo - E_ch).max(axis=1) <= 1e-10 * np.abs(E_ch[:, 0])).all()


def test_compressed_coulomb_rejects_unrestricted():
    P = gen.make_problem_from_geometry(*gen.site_geometry(0), n_occ=(3, 2), n_chol=24, seed=7)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-8, device=0, max_walkers=2, gpu_svd=True)
    with pytest.raises(lo.LoError):
        F.set_coulomb_mode(True)


# ------------------------------------------------------------------------------------------ NEXT-2: multi-determinant trial
def _cas_case(P, n_virt, n_act_occ, n_det, max_exc, n_w, T_svd):
    torch = torch_cuda()
    T = gen.make_cas_trial(P, n_virt=n_virt, n_act_occ=n_act_occ, n_det=n_det, max_exc=max_exc)
    F = lo.Factors.setup(P.h, P.L, [T.C], T_svd, device=0, max_walkers=n_w * n_det, gpu_svd=True)
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w)
    phi = gen.make_walkers(P, n_w)[0]
    E, st = F.local_energy_cas(torch.from_numpy(phi).cuda())
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    Lbar, hbar = oracle.half_rotate(P.L, P.h, T.C)
    n_orb = T.C.shape[1]
    U, sg, W = F.factor_all(0)
    pi, pj = oracle.all_pairs(n_orb)
    fs = oracle.make_factor_set(P.N, n_orb, pi, pj, F.ranks(0), U, sg, W)
    cols = [T.columns(d) for d in range(T.n_det)]
    return T, F, phi, E, st, Lbar, hbar, fs, cols


def test_cas_trial_matches_oracle(c1):
    """lo_local_energy_cas (SMW overlaps / Green's functions, virtual walkers) against the oracle's definition
    (Eq. 12/13: every determinant's own LU, Theta^d and energy) on the library's factor set: all five outputs of every
    walker, 1e-10 relative; 10 determinants (singles and doubles out of the last 3 occupied into 4 virtuals), 7 walkers."""
    T, F, phi, E, st, Lbar, hbar, fs, cols = _cas_case(c1, 4, 3, 10, 2, 7, 1e-4)
    assert (st == 0).all()
    for w in range(phi.shape[0]):
        Eo = np.array(oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi[w]))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])
    # one determinant = the single-determinant path on the reference columns
    F.set_cas_trial(T.n_ref, T.holes[:1], T.parts[:1], T.coef[:1], 7)
    torch = torch_cuda()
    E1d, _ = F.local_energy_cas(torch.from_numpy(phi).cuda())
    F0 = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=7, gpu_svd=True)
    Es, _ = gpu_energy(F0, [phi])
    assert np.abs(E1d.cpu().numpy().T[:, :4] - Es).max() <= 1e-9 * np.abs(Es[:, 0]).max()


def test_cas_trial_triples_and_argument_errors(c0):
    T, F, phi, E, st, Lbar, hbar, fs, cols = _cas_case(c0, 3, 3, 12, 3, 5, 1e-8)
    for w in range(phi.shape[0]):
        Eo = np.array(oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi[w]))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0])
    with pytest.raises(lo.LoError):
        F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, 6)            # 6 * 12 virtual walkers > max_walkers
    bad = T.parts.copy()
    bad[1, 0] = 2                                                        # particle inside the reference
    with pytest.raises(lo.LoError):
        F.set_cas_trial(T.n_ref, T.holes, bad, T.coef, 5)


@pytest.mark.parametrize("cfg,n_virt,n_act,n_det,max_exc,n_w,T_svd", [(1, 4, 3, 10, 2, 7, 1e-4), (0, 3, 3, 12, 3, 5, 1e-8),
                                                                      (1, 5, 6, 40, 4, 19, 1e-3)])
def test_cas_smw_energy_matches_oracle(cfg, n_virt, n_act, n_det, max_exc, n_w, T_svd):
    """LO_CAS_SMW_ENERGY (the rearranged sums of Eq. 21-23: S intermediates once per pair and walker, per-determinant
    bilinear forms) against the oracle's definition with both two-body terms from the factors (Eq. 22), every output of
    every walker, 1e-10 relative; also against the direct-summation mode in compressed-Coulomb mode."""
    torch = torch_cuda()
    P = gen.make_problem(cfg)
    T = gen.make_cas_trial(P, n_virt=n_virt, n_act_occ=n_act, n_det=n_det, max_exc=max_exc)
    F = lo.Factors.setup(P.h, P.L, [T.C], T_svd, device=0, max_walkers=n_w * n_det, gpu_svd=True)
    phi = gen.make_walkers(P, n_w)[0]
    dphi = torch.from_numpy(phi).cuda()
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=True)
    E, st = F.local_energy_cas(dphi)
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    assert (st == 0).all()
    Lbar, hbar = oracle.half_rotate(P.L, P.h, T.C)
    n_orb = T.C.shape[1]
    U, sg, W = F.factor_all(0)
    pi, pj = oracle.all_pairs(n_orb)
    fs = oracle.make_factor_set(P.N, n_orb, pi, pj, F.ranks(0), U, sg, W)
    cols = [T.columns(d) for d in range(T.n_det)]
    for w in range(0, n_w, 3):
        Eo = np.array(oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi[w], compressed_coulomb=True))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])
    F.set_coulomb_mode(True)
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=False)
    Ed, _ = F.local_energy_cas(dphi)
    Ed = Ed.cpu().numpy().T
    assert (np.abs(E - Ed).max(axis=1) <= 1e-9 * np.abs(Ed[:, 0])).all()


@pytest.mark.parametrize("int8", [False, True])
def test_local_energy_is_cuda_graph_capturable(c1, int8):
    """lo_local_energy allocates nothing, does not synchronise and launches only on the caller's stream, so a whole
    step can be captured in a CUDA graph and replayed on new walker data (launch-bound small configs); on both routes (the
    digit slices of the INT8 route are built at the mode switch, before the capture)."""
    torch = torch_cuda()
    n_w = 64
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=n_w, gpu_svd=True)
    F.set_exchange_mode(int8)
    phis = gen.make_walkers(c1, n_w)
    E_ref, _ = gpu_energy(F, phis)
    buf = torch.zeros((n_w, c1.N, c1.n_occ[0]), dtype=torch.complex128, device="cuda")
    E = torch.empty((4, n_w), dtype=torch.complex128, device="cuda")
    st = torch.empty(n_w, dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    import ctypes as C
    with torch.cuda.graph(g, stream=s):
        rc = lo.lib().lo_local_energy(F._h, n_w, C.c_void_p(buf.data_ptr()), None, C.c_void_p(E[0].data_ptr()), C.c_void_p(E[1].data_ptr()),
                                      C.c_void_p(E[2].data_ptr()), C.c_void_p(E[3].data_ptr()), C.c_void_p(st.data_ptr()),
                                      C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == 0
    buf.copy_(torch.from_numpy(phis[0]))
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(E.cpu().numpy().T, E_ref)
    phis2 = gen.make_walkers(c1, n_w, seed=99)
    E2_ref, _ = gpu_energy(F, phis2)
    buf.copy_(torch.from_numpy(phis2[0]))
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(E.cpu().numpy().T, E2_ref)


def test_cas_smw_full_size_sampled_walkers():
    """NEXT-2 at the bench's size: configs[2] in the paper-like (vector) reading, 79 orbitals (73 reference + 6 active
    virtuals), 24 determinants with up to 4 excitations out of 6 active occupied columns, 64 walkers through
    LO_CAS_SMW_ENERGY; two seeded walkers checked against the oracle's definition on the library's factor set."""
    torch = torch_cuda()
    P = gen.make_problem(2, reading="vector")
    T = gen.make_cas_trial(P, n_virt=6, n_act_occ=6, n_det=24, max_exc=4)
    n_w = 64
    F = lo.Factors.setup(P.h, P.L, [T.C], 1e-5, device=0, max_walkers=n_w, gpu_svd=True)
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=True)
    phi = gen.make_walkers(P, n_w)[0]
    E, st = F.local_energy_cas(torch.from_numpy(phi).cuda())
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    assert (st == 0).all() and np.isfinite(E).all()
    Lbar, hbar = oracle.half_rotate(P.L, P.h, T.C)
    n_orb = T.C.shape[1]
    U, sg, W = F.factor_all(0)
    pi, pj = oracle.all_pairs(n_orb)
    fs = oracle.make_factor_set(P.N, n_orb, pi, pj, F.ranks(0), U, sg, W)
    cols = [T.columns(d) for d in range(T.n_det)]
    for w in np.random.default_rng(22).choice(n_w, 2, replace=False):
        Eo = np.array(oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi[w], compressed_coulomb=True))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])


@pytest.mark.parametrize("smw", [False, True])
def test_cas_survey_sizes_200_determinants_rank_6(c1, smw):
    """NEXT-2 at the sizes SURVEY 8(f)-2 names (N_det = 200, excitation rank up to 6, PAPER.md:162 "typically ~ 6", :304-308
    200 determinants): configs[1], 6 active occupied x 6 active virtuals, both modes, 3 walkers, every output against the
    oracle's definition (each determinant's own LU and energy) on the library's factor set, 1e-10.  Ranks 5 and 6 enter the
    k_cas_energy<8> instantiation."""
    torch = torch_cuda()
    n_det, n_w = 200, 3
    T = gen.make_cas_trial(c1, n_virt=6, n_act_occ=6, n_det=n_det, max_exc=6)
    exc = (T.holes >= 0).sum(axis=1)
    assert exc.max() == 6 and (exc == 5).any() and len(set(T.holes[T.holes >= 0].tolist())) == 6
    F = lo.Factors.setup(c1.h, c1.L, [T.C], 1e-3, device=0, max_walkers=n_w * n_det, gpu_svd=True)
    phi = gen.make_walkers(c1, n_w)[0]
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=smw)
    E, st = F.local_energy_cas(torch.from_numpy(phi).cuda())
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    assert (st == 0).all()
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, T.C)
    n_orb = T.C.shape[1]
    U, sg, W = F.factor_all(0)
    pi, pj = oracle.all_pairs(n_orb)
    fs = oracle.make_factor_set(c1.N, n_orb, pi, pj, F.ranks(0), U, sg, W)
    cols = [T.columns(d) for d in range(n_det)]
    for w in range(n_w):
        Eo = np.array(oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi[w], compressed_coulomb=smw))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])


def test_cas_unrestricted_smw_200_determinants_rank_6():
    """The paper's own use of the method -- an open-shell system with a 200-determinant trial, excitation
    rank up to 6 -- through LO_CAS_SMW_ENERGY on an unrestricted factor set: different alpha / beta strings,
    6 active occupied x 6 virtual orbitals per spin, 3 walkers; every output against the oracle's definition (each
    determinant's own LU per spin, w_d = c_d det_a det_b) on the library's factor sets, 1e-10."""
    torch = torch_cuda()
    xyz, fns = gen.site_geometry(1)
    P = gen.make_problem_from_geometry(xyz, fns, (11, 9), 300, seed=41)
    n_det, n_w = 200, 3
    Ta = gen.make_cas_trial(P, n_virt=6, n_act_occ=6, n_det=n_det, max_exc=6, spin=0)
    Tb = gen.make_cas_trial(P, n_virt=6, n_act_occ=6, n_det=n_det, max_exc=6, spin=1)
    assert ((Ta.holes >= 0).sum(axis=1) != (Tb.holes >= 0).sum(axis=1)).any()
    F = lo.Factors.setup(P.h, P.L, [Ta.C, Tb.C], 1e-4, device=0, max_walkers=64, gpu_svd=True)
    F.set_cas_trial(Ta.n_ref, Ta.holes, Ta.parts, Ta.coef, n_w, smw_energy=True)
    F.set_cas_trial_beta(Tb.n_ref, Tb.holes, Tb.parts)
    phis = gen.make_walkers(P, n_w)
    E, st = F.local_energy_cas(torch.from_numpy(phis[0]).cuda(), torch.from_numpy(phis[1]).cuda())
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    assert (st == 0).all()
    hr = [oracle.half_rotate(P.L, P.h, t.C) for t in (Ta, Tb)]
    fss = []
    for s, t in enumerate((Ta, Tb)):
        n_orb = t.C.shape[1]
        U, sg, W = F.factor_all(s)
        pi, pj = oracle.all_pairs(n_orb)
        fss.append(oracle.make_factor_set(P.N, n_orb, pi, pj, F.ranks(s), U, sg, W))
    cols = [[t.columns(d) for d in range(n_det)] for t in (Ta, Tb)]
    for w in range(n_w):
        Eo = np.array(oracle.local_energy_cas_u([Ta.C, Tb.C], cols, Ta.coef, [a for a, _ in hr], [b for _, b in hr], fss,
                                                [phis[0][w], phis[1][w]]))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])


def test_cas_smw_edge_cases(c0):
    """One determinant (no excitation) through the SMW-energy mode = the single-determinant energy with the
    compressed Coulomb term."""
    torch = torch_cuda()
    T = gen.make_cas_trial(c0, n_virt=3, n_act_occ=3, n_det=4, max_exc=2)
    F = lo.Factors.setup(c0.h, c0.L, [T.C], 1e-8, device=0, max_walkers=64, gpu_svd=True)
    phi = gen.make_walkers(c0, 8)[0]
    dphi = torch.from_numpy(phi).cuda()
    F.set_cas_trial(T.n_ref, T.holes[:1], T.parts[:1], T.coef[:1], 8, smw_energy=True)
    E1d, st = F.local_energy_cas(dphi)
    F0 = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=0, max_walkers=8, gpu_svd=True)
    F0.set_coulomb_mode(True)
    Es, _ = gpu_energy(F0, [phi])
    assert np.abs(E1d.cpu().numpy().T[:, :4] - Es).max() <= 1e-9 * np.abs(Es[:, 0]).max()


@pytest.mark.parametrize("n_act,max_exc,n_det", [(9, 2, 40), (12, 4, 60)])
def test_cas_smw_more_than_six_hole_columns(c1, n_act, max_exc, n_det):
    """More than 6 distinct hole columns in LO_CAS_SMW_ENERGY (closed shell): the active set is cut into groups of 3 and the
    S intermediates are formed in one pass per pair of groups (3 groups -> 6 passes, 4 groups -> 10); every output against
    the oracle's definition with both two-body terms from the factors (Eq. 22), 1e-10, and against the direct-summation
    mode.  More than 12 hole columns are refused."""
    torch = torch_cuda()
    n_w = 5
    T = gen.make_cas_trial(c1, n_virt=5, n_act_occ=n_act, n_det=n_det, max_exc=max_exc)
    assert len(set(T.holes[T.holes >= 0].tolist())) == n_act
    F = lo.Factors.setup(c1.h, c1.L, [T.C], 1e-3, device=0, max_walkers=n_w * n_det, gpu_svd=True)
    phi = gen.make_walkers(c1, n_w)[0]
    dphi = torch.from_numpy(phi).cuda()
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=True)
    E, st = F.local_energy_cas(dphi)
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    assert (st == 0).all()
    Lbar, hbar = oracle.half_rotate(c1.L, c1.h, T.C)
    n_orb = T.C.shape[1]
    U, sg, W = F.factor_all(0)
    pi, pj = oracle.all_pairs(n_orb)
    fs = oracle.make_factor_set(c1.N, n_orb, pi, pj, F.ranks(0), U, sg, W)
    cols = [T.columns(d) for d in range(T.n_det)]
    for w in (0, n_w - 1):
        Eo = np.array(oracle.local_energy_cas(T.C, cols, T.coef, Lbar, hbar, fs, phi[w], compressed_coulomb=True))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])
    F.set_coulomb_mode(True)
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=False)
    Ed, _ = F.local_energy_cas(dphi)
    assert (np.abs(E - Ed.cpu().numpy().T).max(axis=1) <= 1e-9 * np.abs(E[:, 0])).all()
    if n_act == 12:
        T13 = gen.make_cas_trial(c1, n_virt=5, n_act_occ=13, n_det=80, max_exc=2)
        assert len(set(T13.holes[T13.holes >= 0].tolist())) == 13
        F13 = lo.Factors.setup(c1.h, c1.L, [T13.C], 1.0, device=0, max_walkers=160, gpu_svd=True)
        with pytest.raises(lo.LoError):
            F13.set_cas_trial(T13.n_ref, T13.holes, T13.parts, T13.coef, 2, smw_energy=True)
        F13.set_cas_trial(T13.n_ref, T13.holes, T13.parts, T13.coef, 2, smw_energy=False)


def test_cas_unrestricted_matches_oracle():
    """Unrestricted multi-determinant trial (different alpha / beta strings, LO_CAS_DIRECT on an n_spin = 2 factor set)
    against the oracle's definition on the library's factor sets: every output of every walker, 1e-10 relative."""
    torch = torch_cuda()
    xyz, fns = gen.site_geometry(1)
    P = gen.make_problem_from_geometry(xyz, fns, (9, 7), 300, seed=31)
    n_det, n_w = 8, 5
    Ta = gen.make_cas_trial(P, n_virt=3, n_act_occ=3, n_det=n_det, max_exc=2, spin=0)
    Tb = gen.make_cas_trial(P, n_virt=4, n_act_occ=2, n_det=n_det, max_exc=2, spin=1)
    F = lo.Factors.setup(P.h, P.L, [Ta.C, Tb.C], 1e-6, device=0, max_walkers=n_w * n_det, gpu_svd=True)
    F.set_cas_trial(Ta.n_ref, Ta.holes, Ta.parts, Ta.coef, n_w)
    phis = gen.make_walkers(P, n_w)
    with pytest.raises(lo.LoError):
        F.local_energy_cas(torch.from_numpy(phis[0]).cuda())                 # beta strings missing
    F.set_cas_trial_beta(Tb.n_ref, Tb.holes, Tb.parts)
    E, st = F.local_energy_cas(torch.from_numpy(phis[0]).cuda(), torch.from_numpy(phis[1]).cuda())
    torch.cuda.synchronize()
    E, st = E.cpu().numpy().T, st.cpu().numpy()
    assert (st == 0).all()
    hr = [oracle.half_rotate(P.L, P.h, t.C) for t in (Ta, Tb)]
    fss = []
    for s, t in enumerate((Ta, Tb)):
        n_orb = t.C.shape[1]
        U, sg, W = F.factor_all(s)
        pi, pj = oracle.all_pairs(n_orb)
        fss.append(oracle.make_factor_set(P.N, n_orb, pi, pj, F.ranks(s), U, sg, W))
    cols = [[t.columns(d) for d in range(n_det)] for t in (Ta, Tb)]
    for w in range(n_w):
        Eo = np.array(oracle.local_energy_cas_u([Ta.C, Tb.C], cols, Ta.coef, [a for a, _ in hr], [b for _, b in hr], fss,
                                                [phis[0][w], phis[1][w]]))
        assert np.abs(E[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, E[w], Eo)
        assert abs(E[w, 4] - Eo[4]) <= TOL * abs(Eo[4])
    # the rearranged SMW energy (Eq. 21-23) for the same unrestricted trial: exchange per spin from the S intermediates, Coulomb
    # by the Cholesky route from SMW-updated X^g (no opposite-spin pair blocks); same oracle, same tolerance
    F.set_cas_trial(Ta.n_ref, Ta.holes, Ta.parts, Ta.coef, n_w, smw_energy=True)
    with pytest.raises(lo.LoError):
        F.local_energy_cas(torch.from_numpy(phis[0]).cuda(), torch.from_numpy(phis[1]).cuda())      # beta strings missing
    F.set_cas_trial_beta(Tb.n_ref, Tb.holes, Tb.parts)
    Es, sts = F.local_energy_cas(torch.from_numpy(phis[0]).cuda(), torch.from_numpy(phis[1]).cuda())
    torch.cuda.synchronize()
    Es, sts = Es.cpu().numpy().T, sts.cpu().numpy()
    assert (sts == 0).all()
    assert (np.abs(Es - E).max(axis=1) <= 1e-9 * np.abs(E[:, 0])).all()
    for w in range(n_w):
        Eo = np.array(oracle.local_energy_cas_u([Ta.C, Tb.C], cols, Ta.coef, [a for a, _ in hr], [b for _, b in hr], fss,
                                                [phis[0][w], phis[1][w]]))
        assert np.abs(Es[w, :4] - Eo[:4]).max() <= TOL * abs(Eo[0]), (w, Es[w], Eo)
        assert abs(Es[w, 4] - Eo[4]) <= TOL * abs(Eo[4])


def test_large_occupation_s1_path():
    """More occupied orbitals than one column block of the overlap kernel holds (O = 200 > 160) and than the
    shared-memory Gauss-Jordan holds (global-workspace variant): Theta against the oracle's LU, E1 / E_J against the
    oracle's Cholesky route.  The threshold truncates every pair away (the pair SVDs still run: 20 100 pairs)."""
    torch = torch_cuda()
    xyz, fns = gen.site_geometry(0)
    P = gen.make_problem_from_geometry(xyz, [52] * 4, (200,), 8, seed=77)
    n_w = 3
    phis = gen.make_walkers(P, n_w)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e9, device=0, max_walkers=n_w, gpu_svd=True)
    assert F.info().sum_rank[0] == 0
    Eg, st = gpu_energy(F, phis)
    assert (st == 0).all()
    th_g = F.theta_host(0, n_w)
    Lbar, hbar = oracle.half_rotate(P.L, P.h, P.psi[0])
    for w in range(n_w):
        th, _, s = oracle.theta(P.psi[0], phis[0][w])
        assert s == 0 and np.abs(th_g[w] - th).max() <= 1e-10 * np.abs(th).max()
        e1, ej = oracle.onebody_coulomb([Lbar], [hbar], [th])
        scale = abs(e1 + ej)
        assert abs(Eg[w, 1] - e1) <= TOL * scale and abs(Eg[w, 2] - ej) <= TOL * scale and Eg[w, 3] == 0


@pytest.mark.parametrize("smw", [False, True])
def test_cas_singular_reference_overlap_is_flagged(c0, smw):
    """A walker with a zero orbital has a singular reference overlap: status 1 and NaN energies for that walker only,
    in both multi-determinant modes; the other walkers are unaffected."""
    torch = torch_cuda()
    T = gen.make_cas_trial(c0, n_virt=3, n_act_occ=3, n_det=6, max_exc=2)
    F = lo.Factors.setup(c0.h, c0.L, [T.C], 1e-8, device=0, max_walkers=24, gpu_svd=True)
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, 4, smw_energy=smw)
    phi = gen.make_walkers(c0, 4)[0].copy()
    E_ok, st_ok = F.local_energy_cas(torch.from_numpy(phi).cuda())
    phi[2, :, 1] = 0.0
    E, st = F.local_energy_cas(torch.from_numpy(phi).cuda())
    torch.cuda.synchronize()
    E, st, E_ok = E.cpu().numpy().T, st.cpu().numpy(), E_ok.cpu().numpy().T
    assert st.tolist() == [0, 0, 1, 0] and np.isnan(E[2]).all()
    ok = [0, 1, 3]
    assert np.array_equal(E[ok], E_ok[ok])


def test_int8_slicing_probe_on_tcgen05():
    """The gated experiment of DESIGN.md 10.1, NOT on the product path: one FP64-accurate 128 x 128 x 384 GEMM
    tile from 6 x 6 signed 7-bit INT8 slices (21 digit products, tcgen05.mma kind::i8 into TMEM, fp64 recombination).  Checked
    here: the result agrees with the fp64 product to 1e-10 of max|C| (the emulation predicts ~2e-11), and the tile takes
    less than 1/1.3 of what the same tile costs on the DMMA pipe at its measured peak (the gate of the experiment)."""
    torch_cuda()
    err = lo.measure_peak("int8_tile_err")
    us = lo.measure_peak("int8_tile_us")
    dmma_tflops = lo.measure_peak("dmma")
    dmma_us = 2.0 * 128 * 128 * 384 / (dmma_tflops * 1e12 / 148) * 1e6          # one SM's share of the measured DMMA peak
    assert err <= 1e-10, err
    assert us * 1.3 <= dmma_us, (us, dmma_us)


# ------------------------------------------------------------------------------------------ exchange from INT8 digit slices (tcgen05)
def int8_energy(F, phis):
    """Energies with lo_set_exchange_mode(LO_EXCHANGE_INT8), two calls (bitwise repeatable), the set left in DMMA mode."""
    F.set_exchange_mode(True)
    try:
        assert F.info().exchange_mode == 1 and F.info().int8_bytes > 0
        Eq, st = gpu_energy(F, phis)
        Eq2, _ = gpu_energy(F, phis)
    finally:
        F.set_exchange_mode(False)
    assert np.array_equal(Eq, Eq2, equal_nan=True), "INT8 exchange: repeated call differs"
    return Eq, st


@pytest.mark.parametrize("cfg,T,n_w", [(0, 1e-8, 8), (1, 1e-6, 256), (1, 1e-4, 70), (1, 1e-6, 1), (1, 5.0, 33)])
def test_exchange_int8_mode_matches_oracle(cfg, T, n_w):
    """lo_set_exchange_mode(LO_EXCHANGE_INT8): the exchange projections AND the Coulomb / one-body contraction X^g_w from 7 x 7
    signed 7-bit digit slices on the tcgen05 tensor cores (28 exact int32 digit products, fp64 recombination).  Every walker and
    every part (E1, E_J, E_K) against the oracle on the library's factor set at the 1e-10 of the default route; ragged walker
    counts (70, 1, 33) and tiles of every height (T = 1e-4: ragged ranks; T = 5: every pair truncated away, Coulomb only)."""
    P = gen.make_problem(cfg)
    phis = gen.make_walkers(P, n_w, seed=7)
    F = lo.Factors.setup(P.h, P.L, P.psi, T, device=0, max_walkers=max(n_w, 64), gpu_svd=True)
    Ed, st = gpu_energy(F, phis)
    Eq, sq = int8_energy(F, phis)
    Eo, _ = oracle_energy(P, F, phis)
    assert (st == 0).all() and (sq == 0).all()
    assert_parity(Eq, Eo)
    assert_close(Eq, Ed, "INT8 route vs DMMA route", tol=1e-10)
    # back in DMMA mode the default result is reproduced bit for bit
    Ed2, _ = gpu_energy(F, phis)
    assert np.array_equal(Ed2, Ed)


@pytest.mark.parametrize("n_w", [5, 130])
def test_propagator_int8_mode_matches_oracle(c1, n_w):
    """lo_propagator in LO_EXCHANGE_INT8 mode (digits of Lt and of the fields, k_coulomb_i8 with one K segment): element by element
    against the oracle's triple loop, 5e-12 of max|B_w| (the digits keep 2^-46 .. 2^-48 of the largest |x^g_w| of the walker and of
    the largest |L^g_pq| of the row, summed over n_chol terms; here with one field component 1000 x the others), on a ragged batch;
    switching back reproduces the DMMA result bit for bit."""
    torch = torch_cuda()
    F = lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=0, max_walkers=n_w, gpu_svd=True, propagator=True)
    rng = np.random.default_rng(12)
    x = rng.standard_normal((n_w, c1.n_chol)) + 1j * rng.standard_normal((n_w, c1.n_chol))
    x[:, 5] *= 1e3                                     # a field component far above the others
    xd = torch.from_numpy(x).cuda()
    F.propagator(xd)
    torch.cuda.synchronize()
    ws = [0, 3, 4] if n_w == 5 else [0, 63, 64, 129]
    Bd = [F.propagator_host(w) for w in ws]
    F.set_exchange_mode(True)
    F.propagator(xd)
    torch.cuda.synchronize()
    for w, B0 in zip(ws, Bd):
        Bo = oracle.propagator(c1.L, x[w])
        Bq = F.propagator_host(w)
        assert np.abs(Bq - Bo).max() <= 5e-12 * np.abs(Bo).max()
        assert np.abs(Bq - B0).max() <= 5e-12 * np.abs(Bo).max()
    F.set_exchange_mode(False)
    F.propagator(xd)
    torch.cuda.synchronize()
    for w, B0 in zip(ws, Bd):
        assert np.array_equal(F.propagator_host(w), B0)


def test_exchange_int8_mode_unrestricted_and_host_variant():
    """Same check for an unrestricted trial (two tile lists, panels of both spins) and through lo_local_energy_host (walker
    chunks of different sizes through the same sliced factor set)."""
    torch = torch_cuda()
    xyz, fns = gen.site_geometry(1)
    P = gen.make_problem_from_geometry(xyz, fns, (9, 7), 300, seed=31)
    phis = gen.make_walkers(P, 200)
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-6, device=0, max_walkers=200, gpu_svd=True)
    Eq, sq = int8_energy(F, phis)
    Eo, _ = oracle_energy(P, F, phis)
    assert (sq == 0).all()
    assert_parity(Eq, Eo)
    F.set_exchange_mode(True)
    Eh, sh = F.local_energy_host([torch.from_numpy(np.ascontiguousarray(p)).pin_memory() for p in phis])
    F.set_exchange_mode(False)
    assert_close(Eh, Eq, "host-buffer variant, INT8 exchange")


def test_exchange_int8_mode_singular_walker_and_errors(c0):
    """A singular walker is flagged and NaN, the others are untouched by it (every walker has its own digit exponents);
    host-only factor sets and unknown modes are refused."""
    torch = torch_cuda()
    phis = gen.make_walkers(c0, 4)
    bad = [p.copy() for p in phis]
    bad[0][2][:, 1] = 0.0                       # a zero orbital: exactly singular overlap
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=0, max_walkers=64)
    Eq, sq = int8_energy(F, bad)
    Eok, _ = int8_energy(F, phis)
    assert sq.tolist() == [0, 0, 1, 0] and np.isnan(Eq[2]).all()
    assert np.array_equal(Eq[[0, 1, 3]], Eok[[0, 1, 3]])
    with pytest.raises(lo.LoError):
        lo._check(lo.lib().lo_set_exchange_mode(F._h, 7))
    Fh = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=-1)
    with pytest.raises(lo.LoError):
        Fh.set_exchange_mode(True)


def test_exchange_int8_mode_c2_full_size(c2_built):
    """BASELINE.json:configs[2] in bench.py's launch configuration with the INT8 exchange: all 512 walkers, 64 seeded walkers
    against the oracle on the library's factor set, every walker against the DMMA route."""
    P, phis, F = c2_built
    Ed, _ = gpu_energy(F, phis)
    Eq, sq = int8_energy(F, phis)
    assert (sq == 0).all() and np.isfinite(Eq).all()
    idx = np.random.default_rng(12).choice(P.n_w, 64, replace=False)
    Eo, _ = oracle_energy(P, F, phis, idx)
    assert_parity(Eq[idx], Eo)
    assert_close(Eq, Ed, "INT8 exchange vs DMMA exchange, configs[2]", tol=1e-10)
