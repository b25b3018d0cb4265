"""Seeded synthetic problems with the shapes of BASELINE.json:configs[0..4].

The paper's workloads are real molecules (dodecane, polyacenes, metallocenes, platonic cages;
PAPER.md:193-310) whose integrals and trials are not available; BASELINE.json replaces them by one
seeded generator ("sites" carrying basis functions and Cholesky vectors, distance-damped random
tensors).  This module implements that generator and nothing else: no Green's function, no
half-rotation, no SVD, no energy.  Readings of the generator's silent points are listed in
DESIGN.md ("Input recipe") and follow SURVEY.md section 8(d).

Random numbers: numpy Philox (counter based), one independent stream per array, keyed by
(seed, tag).  Draw order inside an array is C order of the array as documented per function.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

_TAG_H, _TAG_PSI, _TAG_L, _TAG_PHI, _TAG_ROT = 1, 2, 3, 4, 5
BASE_SEED = 22020832  # arxiv id of the paper; seed of config k is BASE_SEED + k


def _rng(seed: int, tag: int, sub: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[(int(seed) << 8) + tag, sub]))


# ----------------------------------------------------------------------------- geometries
def _line(n, spacing):
    xyz = np.zeros((n, 3))
    xyz[:, 0] = spacing * np.arange(n)
    return xyz


def _ring(n, radius, z=0.0, phase=0.0):
    a = phase + 2 * np.pi * np.arange(n) / n
    return np.stack([radius * np.cos(a), radius * np.sin(a), np.full(n, z)], axis=1)


def _geom_c0():
    # 4 sites on a line, spacing 1.4, 6 functions and 24 Cholesky vectors per site
    return _line(4, 1.4), [6] * 4


def _geom_c1():
    # hexagon of radius 1.4 (= bond 1.4) + 6 outer sites placed radially at +1.1
    ring, outer = _ring(6, 1.4), _ring(6, 2.5)
    return np.concatenate([ring, outer]), [14] * 6 + [5] * 6


def _geom_c2():
    # five linearly fused hexagons, bond 1.4: 22 ring sites; 14 outer sites 1.1 away along the
    # outward bisector of every ring site that has only two ring neighbours
    b = 1.4
    dx = np.sqrt(3.0) * b
    pts = []
    for k in range(5):
        cx = k * dx
        for a in range(6):
            ang = np.pi / 6 + a * np.pi / 3
            pts.append((round(cx + b * np.cos(ang), 9), round(b * np.sin(ang), 9)))
    uniq = sorted(set(pts), key=lambda t: (t[0], t[1]))
    ring = np.array([[x, y, 0.0] for x, y in uniq])
    assert len(ring) == 22
    outer = []
    for s in range(22):
        d = np.linalg.norm(ring - ring[s], axis=1)
        nb = np.where((d > 1e-6) & (d < b * 1.01))[0]
        if len(nb) == 2:
            v = -sum((ring[n] - ring[s]) / np.linalg.norm(ring[n] - ring[s]) for n in nb)
            outer.append(ring[s] + 1.1 * v / np.linalg.norm(v))
    outer = np.array(outer)
    assert len(outer) == 14
    return np.concatenate([ring, outer]), [14] * 22 + [5] * 14


def _geom_c3():
    # two parallel pentagons (radius 1.19, edge 1.4) at z = +-1.65, 10 outer sites radially at +1.1,
    # one central site with 25 functions.  10a+10b = 475 has no integer solution, so ring sites
    # carry 30 functions and outer sites alternate 18/17.
    top, bot = _ring(5, 1.19, 1.65), _ring(5, 1.19, -1.65)
    otop, obot = _ring(5, 2.29, 1.65), _ring(5, 2.29, -1.65)
    xyz = np.concatenate([top, bot, otop, obot, np.zeros((1, 3))])
    return xyz, [30] * 10 + [18, 17] * 5 + [25]


def _geom_c4():
    # closed 3D cage: 140 sites x 5 functions on a Fibonacci sphere whose radius (4.35) gives a
    # nearest-neighbour distance of about 1.4 (site count/radius not given by BASELINE.json)
    n = 140
    k = np.arange(n) + 0.5
    phi = np.arccos(1 - 2 * k / n)
    th = np.pi * (1 + 5 ** 0.5) * k
    r = 4.35
    xyz = np.stack([r * np.cos(th) * np.sin(phi), r * np.sin(th) * np.sin(phi), r * np.cos(phi)], axis=1)
    return xyz, [5] * n


@dataclass(frozen=True)
class ConfigSpec:
    name: str
    geom: object
    n_occ: tuple          # (N_occ,) closed shell or (N_alpha, N_beta) unrestricted
    n_chol: int
    n_w: int
    thresholds: tuple


CONFIGS = {
    0: ConfigSpec("C0 tiny closed-shell chain", _geom_c0, (6,), 96, 8, (1e-8,)),
    1: ConfigSpec("C1 benzene-sized", _geom_c1, (21,), 570, 256, (1e-4, 1e-6)),
    2: ConfigSpec("C2 pentacene-sized", _geom_c2, (73,), 1900, 512, (1e-5,)),
    3: ConfigSpec("C3 open-shell metallocene-sized", _geom_c3, (65, 63), 2500, 1024, (1e-5,)),
    4: ConfigSpec("C4 3D cage cluster", _geom_c4, (130,), 3500, 2048, (1e-3, 1e-4, 1e-5, 1e-6)),
}


def site_geometry(config: int):
    """(xyz [n_sites,3], functions per site) of config k."""
    return CONFIGS[config].geom()


def _chol_per_site(n_chol, fns):
    """N_chol split over sites proportionally to functions per site (largest remainder, ties to
    the lower site index)."""
    fns = np.asarray(fns, dtype=np.int64)
    exact = n_chol * fns / fns.sum()
    base = np.floor(exact).astype(np.int64)
    rem = int(n_chol - base.sum())
    order = sorted(range(len(fns)), key=lambda s: (-(exact[s] - base[s]), s))
    for s in order[:rem]:
        base[s] += 1
    return base


@dataclass
class Problem:
    name: str
    reading: str
    seed: int
    N: int
    n_chol: int
    n_occ: tuple
    site_xyz: np.ndarray
    site_of_fn: np.ndarray
    site_of_chol: np.ndarray
    h: np.ndarray                       # [N,N] symmetric fp64
    L: np.ndarray                       # [n_chol,N,N] fp64, each slice symmetric
    psi: list = field(default_factory=list)   # per spin: [N,n_occ[s]] fp64, orthonormal columns
    n_w: int = 0
    thresholds: tuple = ()

    @property
    def n_spin(self):
        return len(self.n_occ)


def _lowdin(c):
    s = c.T @ c
    w, v = np.linalg.eigh(s)
    return c @ (v * (1.0 / np.sqrt(w))) @ v.T


def chain_geometry(n_sites, fns_per_site=3, spacing=1.4):
    """Extended geometry for the pair-screening study (pairs N^2 -> N): n_sites on a line."""
    xyz = np.zeros((n_sites, 3))
    xyz[:, 0] = spacing * np.arange(n_sites)
    return xyz, [fns_per_site] * n_sites


def make_problem_from_geometry(xyz, fns, n_occ, n_chol, seed, reading="element", name="custom",
                               chol_per_site=None, dtype_L=np.float64) -> Problem:
    """The BASELINE.json generator on an arbitrary site geometry.

    h_pq   = N(0,1) exp(-|R_p-R_q|), drawn for p<=q (row-major upper triangle of an [N,N] draw), mirrored.
    Psi    : per spin an [N,n_occ] standard-normal draw; column i damped by exp(-|R_p-c_i|),
             c_i = site (i mod n_sites); Loewdin-orthonormalised.
    L^g_pq = g exp(-0.8(|R_p-R_g|+|R_q-R_g|)); reading "element": independent g per (gamma,p<=q),
             mirrored (upper triangle of an [N,N] draw per gamma); reading "vector": one g per gamma.
    """
    xyz = np.asarray(xyz, dtype=np.float64)
    fns = list(fns)
    N = int(sum(fns))
    site_of_fn = np.repeat(np.arange(len(fns)), fns)
    cps = _chol_per_site(n_chol, fns) if chol_per_site is None else np.asarray(chol_per_site)
    assert int(cps.sum()) == n_chol
    site_of_chol = np.repeat(np.arange(len(fns)), cps)
    Rp = xyz[site_of_fn]
    dpq = np.linalg.norm(Rp[:, None, :] - Rp[None, :, :], axis=2)

    g = _rng(seed, _TAG_H).standard_normal((N, N))
    h = np.triu(g) * np.exp(-dpq)
    h = h + np.triu(h, 1).T

    psi = []
    for s, no in enumerate(n_occ):
        c = _rng(seed, _TAG_PSI, s).standard_normal((N, no))
        centers = xyz[np.arange(no) % len(fns)]
        damp = np.exp(-np.linalg.norm(Rp[:, None, :] - centers[None, :, :], axis=2))
        psi.append(np.ascontiguousarray(_lowdin(c * damp)))

    L = np.empty((n_chol, N, N), dtype=dtype_L)
    Rg = xyz[site_of_chol]
    dec = np.exp(-0.8 * np.linalg.norm(Rp[None, :, :] - Rg[:, None, :], axis=2))   # [n_chol,N]
    rng = _rng(seed, _TAG_L)
    if reading == "element":
        chunk = max(1, (1 << 24) // (N * N))
        for g0 in range(0, n_chol, chunk):
            g1 = min(n_chol, g0 + chunk)
            gg = rng.standard_normal((g1 - g0, N, N))
            gg = np.triu(gg)
            gg = gg + np.transpose(np.triu(gg, 1), (0, 2, 1))
            L[g0:g1] = gg * dec[g0:g1, :, None] * dec[g0:g1, None, :]
    elif reading == "vector":
        gv = rng.standard_normal(n_chol)
        chunk = max(1, (1 << 24) // (N * N))
        for g0 in range(0, n_chol, chunk):
            g1 = min(n_chol, g0 + chunk)
            L[g0:g1] = gv[g0:g1, None, None] * dec[g0:g1, :, None] * dec[g0:g1, None, :]
    else:
        raise ValueError("reading must be 'element' or 'vector'")
    return Problem(name=name, reading=reading, seed=seed, N=N, n_chol=n_chol, n_occ=tuple(n_occ),
                   site_xyz=xyz, site_of_fn=site_of_fn, site_of_chol=site_of_chol, h=h, L=L, psi=psi)


def make_problem(config: int, seed: int | None = None, reading: str = "element") -> Problem:
    """Problem of BASELINE.json:configs[config] (h, L, Psi); seed defaults to BASE_SEED+config."""
    spec = CONFIGS[config]
    xyz, fns = spec.geom()
    seed = BASE_SEED + config if seed is None else seed
    p = make_problem_from_geometry(xyz, fns, spec.n_occ, spec.n_chol, seed, reading, spec.name)
    p.n_w, p.thresholds = spec.n_w, spec.thresholds
    return p


def make_walkers(problem: Problem, n_w: int | None = None, seed: int | None = None,
                 perturbation: float = 0.1, real: bool = False) -> list:
    """Walkers Phi = Psi + perturbation*(N(0,1)+iN(0,1)), column-normalised; per spin an
    [n_w,N,n_occ] complex128 array (draw: one [n_w,N,n_occ,2] standard-normal block per spin)."""
    n_w = problem.n_w if n_w is None else n_w
    seed = problem.seed if seed is None else seed
    out = []
    for s, psi in enumerate(problem.psi):
        z = _rng(seed, _TAG_PHI, s).standard_normal((n_w,) + psi.shape + (2,))
        phi = psi[None] + perturbation * (z[..., 0] + (0.0 if real else 1j) * z[..., 1])
        phi = phi.astype(np.complex128)
        phi /= np.linalg.norm(phi, axis=1, keepdims=True)
        out.append(np.ascontiguousarray(phi))
    return out


def random_orthogonal(n: int, seed: int) -> np.ndarray:
    """Haar-ish random orthogonal matrix (QR of a normal draw, sign-fixed); used by rotation pins."""
    q, r = np.linalg.qr(_rng(seed, _TAG_ROT).standard_normal((n, n)))
    return q * np.sign(np.diag(r))


_TAG_CAS = 7


@dataclass
class CasTrial:
    """A seeded multi-determinant (CAS-type) trial sum_d c_d |d> of closed-shell determinants (the same excitation in
    both spins), every |d> at most `max_exc` excitations away from the reference: data only."""
    C: np.ndarray        # [N, n_ref + n_virt] orthonormal orbitals: reference occupied first, then active virtuals
    n_ref: int
    holes: np.ndarray    # [n_det, max_exc] int32: replaced column positions of the reference (< n_ref), -1 = unused
    parts: np.ndarray    # [n_det, max_exc] int32: orbital (column of C, >= n_ref) put in that position, -1 = unused
    coef: np.ndarray     # [n_det] fp64 CI coefficients c_d

    @property
    def n_det(self):
        return len(self.coef)

    def columns(self, d):
        """Columns of C occupied in determinant d, in the reference's column positions."""
        cols = np.arange(self.n_ref)
        for hpos, part in zip(self.holes[d], self.parts[d]):
            if hpos >= 0:
                cols[hpos] = part
        return cols


def make_cas_trial(problem: Problem, n_virt: int, n_act_occ: int, n_det: int, max_exc: int, seed: int | None = None,
                   spin: int = 0) -> CasTrial:
    """Reference = problem.psi[0]; `n_virt` active virtuals = Gaussian columns damped like the occupied ones, projected
    onto the complement of the reference and Loewdin-orthonormalised; determinant 0 is the reference (c=1), the others
    replace e in 1..max_exc of the last `n_act_occ` reference columns by distinct virtuals (no duplicates), with
    c_d = 0.3 N(0,1) 2^-e.  `spin` picks problem.psi[spin] (its own random stream): an unrestricted trial is one call per
    spin with the same n_det / max_exc, the alpha call's coefficients being the c_d."""
    seed = problem.seed if seed is None else seed
    rng = _rng(seed, _TAG_CAS, spin)
    psi = problem.psi[spin]
    N, O = psi.shape
    Rp = problem.site_xyz[problem.site_of_fn]
    centers = problem.site_xyz[np.arange(n_virt) % len(problem.site_xyz)]
    damp = np.exp(-np.linalg.norm(Rp[:, None, :] - centers[None, :, :], axis=2))
    v = rng.standard_normal((N, n_virt)) * damp
    v = v - psi @ (psi.T @ v)
    v = _lowdin(v)
    v = v - psi @ (psi.T @ v)          # re-project: keeps C^T C = 1 to rounding
    C = np.ascontiguousarray(np.concatenate([psi, _lowdin(v)], axis=1))
    holes = -np.ones((n_det, max_exc), dtype=np.int32)
    parts = -np.ones((n_det, max_exc), dtype=np.int32)
    coef = np.ones(n_det)
    seen = {()}
    d = 1
    while d < n_det:
        e = int(rng.integers(1, min(max_exc, n_act_occ, n_virt) + 1))
        hs = np.sort(rng.choice(np.arange(O - n_act_occ, O), e, replace=False))
        ps = np.sort(rng.choice(np.arange(O, O + n_virt), e, replace=False))
        key = tuple(hs) + tuple(ps)
        if key in seen:
            continue
        seen.add(key)
        holes[d, :e], parts[d, :e] = hs, ps
        coef[d] = 0.3 * rng.standard_normal() * 0.5 ** e
        d += 1
    return CasTrial(C=C, n_ref=O, holes=holes, parts=parts, coef=coef)
