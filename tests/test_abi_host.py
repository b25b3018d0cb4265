"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol include/lo_afqmc.h declares,
argument errors are reported (no compute without a GPU), and the host side of lo_setup (half-rotation, pair SVD,
truncation, rank sort, padding, tiling, re-truncation) agrees with the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import gen
import oracle
import paper_2202_00832_b200 as lo

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "lo_afqmc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(lo_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(lo.EXPORTS), declared ^ set(lo.EXPORTS)
    L = lo.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert b"sm_100a" in L.lo_version()


def test_argument_errors(c0):
    with pytest.raises(lo.LoError) as e:
        lo.Factors.setup(c0.h, c0.L, c0.psi, -1.0, device=-1)
    assert e.value.status == 1
    with pytest.raises(lo.LoError) as e:
        lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=-1, gpu_svd=True)
    assert e.value.status == 1
    F = lo.Factors.setup(c0.h, c0.L, c0.psi, 1e-8, device=-1, max_walkers=4)
    # no device: the energy call must fail loudly, never fall back to the CPU
    out = np.zeros((4, 4), dtype=np.complex128)
    phi = np.zeros((4, c0.N, 6), dtype=np.complex128)
    st = lo.lib().lo_local_energy_host(F._h, 4, phi.ctypes.data, None, out.ctypes.data, None, None)
    assert st == 3 and b"no CPU path" in lo.lib().lo_last_error()
    st = lo.lib().lo_local_energy(F._h, 4, phi.ctypes.data, None, out.ctypes.data, None, None, None, None, None)
    assert st == 3
    with pytest.raises(lo.LoError):
        F.retruncate(1e-9)          # tighter than the original threshold


@pytest.fixture(scope="module")
def c1_host(c1):
    return lo.Factors.setup(c1.h, c1.L, c1.psi, 1e-4, device=-1, max_walkers=8)


def test_host_factors_match_oracle(c1, c1_host):
    info = c1_host.info()
    O, N = c1.n_occ[0], c1.N
    assert (info.N, info.N_pad, info.n_chol, info.n_spin, info.n_pairs[0]) == (N, 128, 570, 1, O * (O + 1) // 2)
    Lbar, _ = oracle.half_rotate(c1.L, c1.h, c1.psi[0])
    pi, pj = oracle.all_pairs(O)
    sel = np.arange(0, len(pi), 9)
    Ut, s, Wt = oracle.full_svd_pairs(Lbar, pi[sel], pj[sel])
    ranks = c1_host.ranks()
    assert info.sum_rank[0] == ranks.sum() and info.max_rank == ranks.max() and info.min_rank == ranks.min()
    assert info.sum_rank_padded == ((ranks + 7) // 8 * 8).sum()
    for n, k in enumerate(sel):
        r_or = int((s[n] > 1e-4).sum())
        assert ranks[k] == r_or
        U, sg, W = c1_host.factor_pair(0, int(pi[k]), int(pj[k]))
        assert np.abs(sg - s[n, :r_or]).max() <= 1e-12 * s[n, 0]
        Y = oracle.pair_eri(Lbar, pi[k], pj[k])
        assert np.abs((U.T * sg) @ W - (Ut[n, :r_or].T * s[n, :r_or]) @ Wt[n, :r_or]).max() <= 1e-11 * s[n, 0]
        assert np.abs((U.T * sg) @ W - Y).max() <= 2 * max(s[n, r_or] if r_or < N else 0, 1e-12 * s[n, 0])
        assert np.abs(U @ U.T - np.eye(r_or)).max() < 1e-12 and np.abs(W @ W.T - np.eye(r_or)).max() < 1e-12


def lapack_pin(F, spin, Lbar, pairs, T, N):
    """Pins the LIBRARY's factors of the listed pairs to LAPACK (numpy.linalg.svd of Y^{ij} = Lbar_i^T Lbar_j formed by
    numpy; none of the repo's SVD routines, oracle or product, takes part): singular values to 1e-12 sigma_1, rank =
    #(sigma > T) except where |sigma - T| <= 1e-10 sigma_max (DESIGN R13), truncated reconstruction U^T sigma W to
    1e-11 sigma_1, orthonormal rows.  Returns the number of pairs whose rank sat inside the ambiguity band."""
    ranks = F.ranks(spin)
    O = int(round((np.sqrt(8 * len(ranks) + 1) - 1) / 2))
    band = 0
    for (i, j) in pairs:
        k = i * O - i * (i - 1) // 2 + (j - i)
        Y = Lbar[:, i, :].T @ Lbar[:, j, :]                      # Y^{ij}_pq = sum_g Lbar^g_ip Lbar^g_jq
        Ul, sl, Wl = np.linalg.svd(Y)
        r_l = int((sl > T).sum())
        r = int(ranks[k])
        if r != r_l:
            lo_, hi = min(r, r_l), max(r, r_l)
            assert (np.abs(sl[lo_:hi] - T) <= 1e-10 * sl[0]).all(), (i, j, r, r_l)
            band += 1
        U, sg, W = F.factor_pair(spin, i, j)
        assert sg.shape == (r,) and (np.diff(sg) <= 0).all()
        assert np.abs(sg - sl[:r]).max(initial=0.0) <= 1e-12 * sl[0], (i, j)
        rec_lib = (U.T * sg) @ W
        rec_lap = (Ul[:, :r] * sl[:r]) @ Wl[:r]
        assert np.abs(rec_lib - rec_lap).max(initial=0.0) <= 1e-11 * sl[0], (i, j)
        if r:
            assert np.abs(U @ U.T - np.eye(r)).max() < 1e-12 and np.abs(W @ W.T - np.eye(r)).max() < 1e-12, (i, j)
    return band


def test_host_factors_pinned_to_lapack(c1, c1_host):
    """All 231 pair blocks of configs[1] (T = 1e-4), host setup path, against LAPACK."""
    O = c1.n_occ[0]
    Lbar = np.einsum("gpq,qi->gip", c1.L, c1.psi[0])             # PAPER.md:127, typed with numpy
    band = lapack_pin(c1_host, 0, Lbar, [(i, j) for i in range(O) for j in range(i, O)], 1e-4, c1.N)
    assert band <= 2


def test_host_factors_low_rank_pinned_to_lapack():
    """Rank-deficient blocks ("vector" reading: rank <= number of sites, the rest of the spectrum is rounding noise) and an
    unrestricted set: the null space must neither be kept nor disturb the kept vectors."""
    xyz, fns = gen.site_geometry(1)
    P = gen.make_problem_from_geometry(xyz, fns, (9, 7), 200, seed=11, reading="vector")
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-6, device=-1, max_walkers=4)
    for s in range(2):
        O = P.n_occ[s]
        Lbar = np.einsum("gpq,qi->gip", P.L, P.psi[s])
        assert F.ranks(s).max() <= len(xyz)
        lapack_pin(F, s, Lbar, [(i, j) for i in range(O) for j in range(i, O)], 1e-6, P.N)


def test_factor_all_order_and_tiles(c1_host, c1):
    U, s, W = c1_host.factor_all()
    ranks = c1_host.ranks()
    off = np.concatenate([[0], np.cumsum(ranks)])
    O = c1.n_occ[0]
    k = 3 * O - 3 + 5 - 3                     # pair (3,5)
    Up, sp, Wp = c1_host.factor_pair(0, 3, 5)
    assert np.array_equal(U[off[k]:off[k + 1]], Up) and np.array_equal(s[off[k]:off[k + 1]], sp)
    info = c1_host.info()
    # every pair is cut into ceil(r_pad/64) row tiles of near-equal size
    assert info.n_tiles == (((ranks + 7) // 8 + 7) // 8).sum()


def test_retruncate_is_prefix(c1_host):
    T2 = 2.0
    F2 = c1_host.retruncate(T2)
    r1, r2 = c1_host.ranks(), F2.ranks()
    assert (r2 <= r1).all() and r2.sum() < r1.sum()
    for (i, j) in [(0, 0), (2, 7), (20, 20)]:
        U1, s1, W1 = c1_host.factor_pair(0, i, j)
        U2, s2, W2 = F2.factor_pair(0, i, j)
        r = len(s2)
        assert r == int((s1 > T2).sum())
        assert np.array_equal(U2, U1[:r]) and np.array_equal(s2, s1[:r]) and np.array_equal(W2, W1[:r])
    assert F2.info().threshold == T2


def test_unrestricted_and_zero_rank_pairs():
    xyz, fns = gen.site_geometry(0)
    P = gen.make_problem_from_geometry(xyz, fns, (5, 3), 30, seed=5, reading="vector")
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-3, device=-1, max_walkers=4)
    info = F.info()
    assert info.n_spin == 2 and tuple(info.n_pairs) == (15, 6)
    ra, rb = F.ranks(0), F.ranks(1)
    assert ra.max() <= 4 and rb.max() <= 4            # "vector" reading: rank <= number of sites
    Fbig = F.retruncate(1e6)                           # everything truncated away
    assert Fbig.info().sum_rank[0] == 0 and Fbig.info().n_tiles == 0
    hr = oracle.half_rotate(P.L, P.h, P.psi[1])
    U, s, W = F.factor_pair(1, 0, 2)
    Y = oracle.pair_eri(hr[0], 0, 2)
    assert np.abs((U.T * s) @ W - Y).max() < 2e-3


def test_walker_shard():
    from paper_2202_00832_b200.dist import walker_shard
    for n, world in [(512, 2), (7, 3), (1, 4), (0, 2)]:
        spans = [walker_shard(n, r, world) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
        sizes = [b - a for a, b in spans]
        assert max(sizes) - min(sizes) <= 1


def _chain_problem():
    xyz, fns = gen.chain_geometry(24, 3)
    return gen.make_problem_from_geometry(xyz, fns, (24,), 120, seed=3)


def test_prescreen_is_bit_identical_and_counts_pairs():
    """The rigorous pre-SVD pair screen (LO_SETUP flag off/on) on a 24-site chain, host setup path: identical ranks, factor
    rows, singular values and tile count; lo_info counts the pairs that were never decomposed; every screened pair has a
    LAPACK sigma_1 <= T (so Eq. 18 gives it rank 0 anyway) and the oracle's bound says the same."""
    P = _chain_problem()
    T = 1e-5
    Fs = lo.Factors.setup(P.h, P.L, P.psi, T, device=-1, max_walkers=4)
    Fn = lo.Factors.setup(P.h, P.L, P.psi, T, device=-1, max_walkers=4, prescreen=False)
    i_s, i_n = Fs.info(), Fn.info()
    assert i_n.n_pairs_prescreened == 0 and i_s.n_pairs_prescreened >= 20
    assert np.array_equal(Fs.ranks(), Fn.ranks()) and i_s.n_tiles == i_n.n_tiles and i_s.sum_rank_padded == i_n.sum_rank_padded
    for a, b in zip(Fs.factor_all(), Fn.factor_all()):
        assert np.array_equal(a, b)
    Lbar, _ = oracle.half_rotate(P.L, P.h, P.psi[0])
    pi, pj = oracle.all_pairs(24)
    fro, tri, _ = oracle.pair_norm_bounds(Lbar, pi, pj)
    assert i_s.n_pairs_prescreened == int((fro <= T).sum()) and int((tri <= T).sum()) <= i_s.n_pairs_prescreened
    s1 = np.array([np.linalg.svd(Lbar[:, i, :].T @ Lbar[:, j, :], compute_uv=False)[0] for i, j in zip(pi, pj)])
    assert (Fs.ranks()[fro <= T] == 0).all() and (s1[fro <= T] <= T).all()
    # the number of kept pairs grows like the chain length, not its square
    kept = []
    for n_sites in (12, 24):
        xyz, fns = gen.chain_geometry(n_sites, 3)
        Pc = gen.make_problem_from_geometry(xyz, fns, (n_sites,), 5 * n_sites, seed=3)
        Fc = lo.Factors.setup(Pc.h, Pc.L, Pc.psi, 1e-3, device=-1, max_walkers=4)
        kept.append(int((Fc.ranks() > 0).sum()))
    assert kept[1] < 3.0 * kept[0] and kept[1] / 300.0 < kept[0] / 78.0        # doubling the chain: pairs x3.85, kept pairs < x3


def test_energy_screen_matches_oracle_rule():
    """lo_screen_pairs against the oracle's plain-loop rule on the library's own factors: the same pairs are dropped, the
    kept rows are untouched, the recorded bound is cK sum_dropped m_ij sigma_1; cutoff 0 is the identity."""
    P = _chain_problem()
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-7, device=-1, max_walkers=4)
    pi, pj = oracle.all_pairs(24)
    U, sg, W = F.factor_all()
    fs = oracle.make_factor_set(P.N, 24, pi, pj, F.ranks(), U, sg, W)
    F0 = F.screen_pairs(0.0)
    assert np.array_equal(F0.ranks(), F.ranks()) and F0.info().n_pairs_energy_screened == 0
    for cutoff in (1e-5, 1e-2, 1.0):
        Fc = F.screen_pairs(cutoff)
        fso, drop, ms1 = oracle.screen_pairs(fs, cutoff)
        assert np.array_equal(Fc.ranks(), fso.r) and 0 < drop.sum() < len(pi)
        Uc, sc, Wc = Fc.factor_all()
        assert np.array_equal(Uc, fso.U) and np.array_equal(sc, fso.sigma) and np.array_equal(Wc, fso.W)
        ic = Fc.info()
        assert ic.n_pairs_energy_screened == int(drop.sum()) and ic.energy_screen_cutoff == cutoff
        assert abs(ic.energy_screen_bound - ms1[drop].sum()) <= 1e-12 * ms1[drop].sum()
    with pytest.raises(lo.LoError):
        F.screen_pairs(-1.0)


def test_randomized_svd_setup_host_path():
    """LO_SETUP_RANDOMIZED_SVD on the host path.  Rank-deficient blocks ("vector"
    reading: rank <= 12 sites, sketch of 16 rows): every non-screened block is accepted, and the factors pass the same
    LAPACK pin as the full method's (singular values 1e-12 sigma_1, ranks, truncated reconstructions, orthonormal rows).
    Full-rank blocks ("element" reading): the a-posteriori check rejects every sketch and the full method's factor set
    comes out bit for bit."""
    xyz, fns = gen.site_geometry(1)
    P = gen.make_problem_from_geometry(xyz, fns, (9,), 200, seed=11, reading="vector")
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-6, device=-1, max_walkers=4, rsvd=16)
    info = F.info()
    assert info.rsvd_sketch == 16 and info.n_pairs_rsvd + info.n_pairs_prescreened == info.n_pairs[0] == 45
    Lbar = np.einsum("gpq,qi->gip", P.L, P.psi[0])
    lapack_pin(F, 0, Lbar, [(i, j) for i in range(9) for j in range(i, 9)], 1e-6, P.N)
    Ff = lo.Factors.setup(P.h, P.L, P.psi, 1e-6, device=-1, max_walkers=4)
    assert np.array_equal(F.ranks(), Ff.ranks())
    Pe = gen.make_problem_from_geometry(xyz, fns, (5,), 200, seed=11)
    Fe = lo.Factors.setup(Pe.h, Pe.L, Pe.psi, 1e-6, device=-1, max_walkers=4, rsvd=16)
    Fe0 = lo.Factors.setup(Pe.h, Pe.L, Pe.psi, 1e-6, device=-1, max_walkers=4)
    assert Fe.info().n_pairs_rsvd == 0
    for a, b in zip(Fe.factor_all(), Fe0.factor_all()):
        assert np.array_equal(a, b)
