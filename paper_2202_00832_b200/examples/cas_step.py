"""One multi-determinant local-energy step on configs[2] in the paper-like "vector" reading:
python -m paper_2202_00832_b200.examples.cas_step N_DET N_WALKERS [direct|smw].  Used for the ncu captures in profiles/."""
import sys

import torch

import gen
import paper_2202_00832_b200 as lo


def main():
    n_det, n_w = int(sys.argv[1]), int(sys.argv[2])
    smw = (sys.argv[3] if len(sys.argv) > 3 else "smw") == "smw"
    P = gen.make_problem(2, reading="vector")
    T = gen.make_cas_trial(P, n_virt=6, n_act_occ=6, n_det=n_det, max_exc=4)
    F = lo.Factors.setup(P.h, P.L, [T.C], 1e-5, device=0, max_walkers=n_w if smw else n_w * n_det, gpu_svd=True)
    F.set_cas_trial(T.n_ref, T.holes, T.parts, T.coef, n_w, smw_energy=smw)
    phi = torch.from_numpy(gen.make_walkers(P, n_w)[0]).cuda()
    for _ in range(3):
        E, st = F.local_energy_cas(phi)
    torch.cuda.synchronize()
    info = F.info()
    print("tiles %d, sum_rank %d, E_L[0] = %s, status ok = %s" % (info.n_tiles, info.sum_rank[0], E[0, 0].item(), bool((st == 0).all())))


if __name__ == "__main__":
    main()
