"""lo_theta_noalloc: the allocation-free S1 entry point (scratch in a file-scope static __device__ array of 4 MiB) against the
ordinary path (lo_local_energy's S1, read back with lo_theta_host).  In a file of its own that pytest collects last."""
import numpy as np
import pytest

import gen
import paper_2202_00832_b200 as lo

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _theta_from_panels(buf, n_w, N):
    """[O][ld_w][N_pad] fp64 panels -> complex [n_w][N][O]"""
    b = buf.cpu().numpy()
    th = b[:, 0:2 * n_w:2, :N] + 1j * b[:, 1:2 * n_w:2, :N]          # [O][n_w][N]
    return np.ascontiguousarray(th.transpose(1, 2, 0))


def test_theta_noalloc_matches_the_ordinary_path_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    P = gen.make_problem(1)                                             # N = 114, n_occ = 21
    N, O = P.N, P.n_occ[0]
    n_max = 200
    assert 16 * n_max * O * O <= lo.LO_NOALLOC_SCRATCH_BYTES
    F = lo.Factors.setup(P.h, P.L, P.psi, 1e-4, device=0, max_walkers=n_max)
    lo.theta_noalloc_init(0)
    psi = torch.from_numpy(np.ascontiguousarray(P.psi[0])).cuda()
    N_pad = (N + 15) // 16 * 16
    out = torch.full((O, 2 * n_max, N_pad), float("nan"), dtype=torch.float64, device="cuda")    # all buffers exist before the calls
    status = torch.full((n_max,), -1, dtype=torch.int32, device="cuda")
    # two calls in a row on the shared scratch: 200 walkers, then 70 other walkers (the scratch still holds the first call's
    # matrices), the second batch with one singular walker
    for n_w, seed, singular in ((200, 5, None), (70, 6, 3)):
        phis = gen.make_walkers(P, n_w, seed=seed)
        if singular is not None:
            phis[0][singular, :, 1] = 0.0
        d = torch.from_numpy(np.ascontiguousarray(phis[0])).cuda()
        F.local_energy([d])
        ref = F.theta_host(0, n_w)
        st_ref = F.local_energy([d])[4].cpu().numpy()
        out.fill_(float("nan"))
        status.fill_(-1)
        mem0 = torch.cuda.mem_get_info()[0]
        lo.theta_noalloc(psi, d, out, status)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == mem0, "lo_theta_noalloc changed the free device memory"
        th = _theta_from_panels(out, n_w, N)
        st = status.cpu().numpy()[:n_w]
        assert np.array_equal(st, st_ref)
        ok = st == 0
        assert ok.sum() == n_w - (0 if singular is None else 1)
        scale = np.abs(ref[ok]).max(axis=(1, 2), keepdims=True)
        assert (np.abs(th[ok] - ref[ok]) / scale).max() <= TOL
        if singular is not None:
            assert np.isnan(th[singular]).all()
        # padding rows p in [N, N_pad) are zeros, rows of walkers beyond n_w untouched
        assert (out[:, :2 * n_w, N:].cpu().numpy()[:, np.repeat(ok, 2)] == 0).all()
        assert torch.isnan(out[:, 2 * n_w:, :]).all()
        assert (status[n_w:] == -1).all()
    F.free()


def test_theta_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    N, O = 114, 21
    n_w = lo.LO_NOALLOC_SCRATCH_BYTES // (16 * O * O) + 1
    psi = torch.zeros((N, O), dtype=torch.float64, device="cuda")
    phi = torch.zeros((n_w, N, O), dtype=torch.complex128, device="cuda")
    out = torch.zeros((O, 2 * n_w, 128), dtype=torch.float64, device="cuda")
    status = torch.zeros((n_w,), dtype=torch.int32, device="cuda")
    with pytest.raises(lo.LoError, match="split the batch"):
        lo.theta_noalloc(psi, phi, out, status)
    with pytest.raises(lo.LoError):
        lo._check(lo.lib().lo_theta_noalloc(0, N, O, 4, psi.data_ptr(), phi.data_ptr(), out.data_ptr(), 7, status.data_ptr(), None))   # odd ld_w
