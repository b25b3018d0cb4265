// lo_cas.cu -- multi-determinant (CAS-type) trial: Sherman-Morrison-Woodbury overlaps and Green's
// functions of the excited determinants (Eq. 20), the direct summation over determinants on virtual walkers (Eq. 12/13)
// and the rearranged SMW energy of Eq. 21-23 (k_cas_pairs, k_cas_H, k_cas_energy, k_cas_e1sum).
#include "lo_device.cuh"

namespace lo {

namespace {

// ------------------------------------------------------------------------------------------------ NEXT-2: multi-determinant trial
// Sherman-Morrison-Woodbury update of the reference (Eq. 20): determinant d replaces the reference columns
// h_1..h_e by the orbitals p_1..p_e, A_d = A + U V^T.  With T = C_virt^T Theta0 (Theta0 = Phi A^-1) and T_d = T[p_k, h_l]:
//   det A_d / det A = det T_d,      Theta^d = Theta0 (I - E_h T_d^-1 (T[p,:] - I[h,:])),
// so in orbital-indexed panels (x = orbital of the factor set, zero when d does not occupy x)
//   Theta^d_x = [x reference, not a hole] Theta0_x + sum_k G_d[k][x] Theta0_{h_k},
//   G_d[k][x] = -sum_l (T_d^-1)_kl T[p_l][x]  (x reference, not a hole),  (T_d^-1)_km  (x = p_m),  0 otherwise.
// k_cas_T: T[w][v][a] = sum_p C[p][n_ref+v] Theta0[a][w][p]; grid n_w, one warp per (v,a), lanes over p.
__global__ void __launch_bounds__(256) k_cas_T(const double* __restrict__ C, int ldc, const double* __restrict__ th0, double2* __restrict__ T,
                                               int N, int N_pad, int n_ref, int n_virt, int ldw0) {
    const int w = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int e = warp; e < n_virt * n_ref; e += 8) {
        const int v = e / n_ref, a = e - v * n_ref;
        const double* re = th0 + ((size_t)a * ldw0 + 2 * w) * N_pad;
        const double* im = re + N_pad;
        double sr = 0.0, si = 0.0;
        for (int p = lane; p < N; p += 32) {
            const double c = C[(size_t)p * ldc + n_ref + v];
            sr = fma(c, re[p], sr);
            si = fma(c, im[p], si);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { sr += __shfl_xor_sync(0xffffffffu, sr, o); si += __shfl_xor_sync(0xffffffffu, si, o); }
        if (lane == 0) T[((size_t)w * n_virt + v) * n_ref + a] = make_double2(sr, si);
    }
}

// ---- NEXT-2, rearranged SMW energy (Eq. 21-23).  Every Theta^d column is a combination of the
// reference column and the active (hole) columns of Theta0, so for pair (x <= y) the projections of U^{xy}, W^{xy} onto the
// panel set P = [x, y, A_1..A_na] of Theta0 ("Q_L^int = U Phi A_act^-1") serve ALL determinants.  They are
// contracted over the singular index K at once,
//     S_t[c][c'] = sum_{K in tile t} wgt_K (U_K . Theta0_c)(W_K . Theta0_c'),     c, c' in P,
// and a determinant's pair energies are small bilinear forms in S (k_cas_energy).  Work item = (row tile, block of 16
// walkers); work units (row fragment, column tile of 4 walkers) dealt evenly to the consumer warps; same TMA/mbarrier pipeline.
constexpr int CP_STAGES = 4;
template <int NP>
struct CpCfg {
    static constexpr int STAGE_BYTES = 2 * EX_BM * 128 + NP * 32 * 128;      // U, W (<= 64 rows) + NP panels x 16 walkers
    static constexpr int SL = NP * NP + 1;      // slice stride (double2) of one (warp, walker): odd, so the 8 lanes of a
                                                // 128-bit shared access land on distinct 16-byte bank groups
    static constexpr int SMEM = CP_STAGES * STAGE_BYTES + 1024 + 128 + EX_RING * 16 + 8 * 4 * SL * 16;
};

// K loop of one (<= 4-fragment) tile for a warp that owns NFW <= 2 row fragments (fg, fg + 2) and one column tile (4
// walkers): both projections of every fragment onto all NP panels; no padding MMAs (instantiated per NFW).
template <int NP, int NFW>
__device__ __forceinline__ void cp_kloop(int KT, uint32_t sbase, uint32_t full, uint32_t empty, int& cslot, uint32_t& cphase, int lane,
                                         const uint32_t (&xo)[4], uint32_t u_row, uint32_t p_row, double (&accU)[2][NP][2],
                                         double (&accW)[2][NP][2]) {
    constexpr int STAGE = CpCfg<NP>::STAGE_BYTES;
    for (int kt = 0; kt < KT; ++kt) {
        if (kt) mbar_wait(full + 8 * cslot, cphase);
        if constexpr (NFW == 0) {
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + 8 * cslot);
        } else {
            const uint32_t st = sbase + cslot * STAGE;
#pragma unroll
            for (int ks = 0; ks < KTILE / 4; ++ks) {
                double a[NFW], w[NFW], bb[NP];
#pragma unroll
                for (int j = 0; j < NFW; ++j) {
                    a[j] = lds_f64(st + u_row + j * 2048 + xo[ks]);
                    w[j] = lds_f64(st + u_row + EX_BM * 128 + j * 2048 + xo[ks]);
                }
#pragma unroll
                for (int c = 0; c < NP; ++c) bb[c] = lds_f64(st + p_row + c * 4096 + xo[ks]);
                if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                for (int j = 0; j < NFW; ++j)
#pragma unroll
                    for (int c = 0; c < NP; ++c) {
                        mma884(accU[j][c][0], accU[j][c][1], a[j], bb[c]);
                        mma884(accW[j][c][0], accW[j][c][1], w[j], bb[c]);
                    }
            }
        }
        if (++cslot == CP_STAGES) { cslot = 0; cphase ^= 1; }
    }
}

template <int NP>
__global__ void __launch_bounds__(384, 1) k_cas_pairs(const __grid_constant__ TmSet tmUs, const __grid_constant__ TmSet tmWs,
                                                      const __grid_constant__ CUtensorMap tmT0, const double* __restrict__ wgt,
                                                      const ExTile* __restrict__ tiles4, const CasPair* __restrict__ pairs, long long n_items,
                                                      int WB, int N_pad, int ldw0, const int* __restrict__ act /* [NP-2] */,
                                                      double2* __restrict__ S, int n_w,
                                                      int pan_base /* first orbital of this spin in the factor set's numbering */) {
    constexpr int STAGE = CpCfg<NP>::STAGE_BYTES;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const uint32_t full = sbase + CP_STAGES * STAGE, empty = full + 8 * CP_STAGES;
    ExTile* ring = reinterpret_cast<ExTile*>(sgen + CP_STAGES * STAGE + 128);
    double2* Sacc = reinterpret_cast<double2*>(sgen + CP_STAGES * STAGE + 128 + EX_RING * 16);     // [8 warps][4 walkers][SL]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KT = N_pad / KTILE;
    if (tid == 0) {
        for (int k = 0; k < 8; ++k) { prefetch_tmap(&tmUs.m[k]); prefetch_tmap(&tmWs.m[k]); }
        prefetch_tmap(&tmT0);
        for (int i = 0; i < CP_STAGES; ++i) { mbar_init(full + 8 * i, 1); mbar_init(empty + 8 * i, 8); }
        fence_barrier_init();
    }
    __syncthreads();
    if (warp < 4) {
        reg_dec_producer();
        if (warp == 0 && lane == 0) {
            int pan[NP];
#pragma unroll
            for (int c = 2; c < NP; ++c) pan[c] = act[c - 2];
            int slot = 0, n = 0;
            uint32_t phase = 0;
            for (long long q = blockIdx.x; q < n_items; q += gridDim.x) {
                const CasPair pr = pairs[q / WB];
                const int wb = (int)(q % WB);
                pan[0] = pr.pi - pan_base;
                pan[1] = pr.pj - pan_base;
                for (int ts = 0; ts < pr.nt; ++ts, ++n) {         // the pair's tiles, one after the other
                    const ExTile tile = tiles4[pr.t0 + ts];
                    const uint32_t tx = (uint32_t)(2 * tile.nfrag * 8 + NP * 32) * 128;
                    for (int kt = 0; kt < KT; ++kt) {
                        mbar_wait(empty + 8 * slot, phase ^ 1);
                        if (kt == 0) ring[n % EX_RING] = tile;
                        const uint32_t st = sbase + slot * STAGE, bar = full + 8 * slot;
                        const int k0 = kt * KTILE;
                        mbar_expect_tx(bar, tx);
                        tma_load_2d(st, &tmUs.m[tile.nfrag - 1], k0, tile.row0, bar);
                        tma_load_2d(st + EX_BM * 128, &tmWs.m[tile.nfrag - 1], k0, tile.row0, bar);
#pragma unroll
                        for (int c = 0; c < NP; ++c)        // 32 real rows (16 walkers) of panel c
                            tma_load_2d(st + 2 * EX_BM * 128 + c * 4096, &tmT0, k0, pan[c] * ldw0 + wb * 32, bar);
                        if (++slot == CP_STAGES) { slot = 0; phase ^= 1; }
                    }
                }
            }
        }
        return;
    }
    reg_inc_consumer();
    // Work item = (pair, block of 16 walkers); its tiles (<= 4 fragments each) run one after the other and S is summed over
    // them in registers, so S exists once per PAIR.  Work units of a tile = (row fragment, column tile of 4 walkers) =
    // 4 * nfrag <= 16; consumer warp cw owns column tile cw & 3 and the fragments (cw >> 2), (cw >> 2) + 2: the two warps
    // of a scheduler (cw, cw + 4) hold nfrag units between them whatever nfrag is, so the four tensor pipes carry equal
    // loads (round 1 dealt (fragment, column half) units of an 8-walker item: 3/3/2/2 over the schedulers at 5 fragments).
    const int cw = warp - 4, g = lane >> 2, t = lane & 3, ctid = tid - 128;
    const int nt = cw & 3, fg = cw >> 2;
    double accU[2][NP][2], accW[2][NP][2];
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int c = 0; c < NP; ++c) accU[j][c][0] = accU[j][c][1] = accW[j][c][0] = accW[j][c][1] = 0.0;
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t u_row = (uint32_t)(fg * 8 + g) * 128;
    const uint32_t p_row = (uint32_t)(2 * EX_BM * 128) + (uint32_t)(nt * 8 + g) * 128;
    constexpr int SL = CpCfg<NP>::SL;
    const bool b0 = g & 1, b1 = g & 2, b2 = g & 4;
    const int c2own = (b0 ? 4 : 0) + (b1 ? 2 : 0) + (b2 ? 1 : 0);
    int cslot = 0, n = 0;
    uint32_t cphase = 0;
    for (long long q = blockIdx.x; q < n_items; q += gridDim.x) {
        const int wb = (int)(q % WB);
        const long long pix = q / WB;
        const int n_sub = pairs[pix].nt;
        double2 sc[NP];                      // this lane's S[c][c2own] of walker 4 nt + t, summed over the pair's rows
#pragma unroll
        for (int c = 0; c < NP; ++c) sc[c] = make_double2(0.0, 0.0);
        for (int ts = 0; ts < n_sub; ++ts, ++n) {
            mbar_wait(full + 8 * cslot, cphase);
            const ExTile tile = ring[n % EX_RING];
            const int nfw = tile.nfrag > fg ? (tile.nfrag - fg + 1) >> 1 : 0;     // warp-uniform, <= 2
            switch (nfw) {
                case 0: cp_kloop<NP, 0>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, p_row, accU, accW); break;
                case 1: cp_kloop<NP, 1>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, p_row, accU, accW); break;
                default: cp_kloop<NP, 2>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, p_row, accU, accW); break;
            }
            // S[c][c'] of the 4 walkers of this warp's column tile.  For every panel c the lane holds the 8 complex products
            // of its own row g (c' = 0..7, zero beyond NP); a transposing butterfly over the 8 row groups (each round sends
            // half of the values and keeps the other half: 8+4+2 exchanges instead of 3 per value) leaves the row sum of
            // column c' = 4 b0 + 2 b1 + b2 (bits of g) in lane g.
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (j >= nfw) break;                     // warp-uniform
                const double wv = __ldg(wgt + tile.row0 + (fg + 2 * j) * 8 + g);
#pragma unroll
                for (int c = 0; c < NP; ++c) {
                    const double ur = wv * accU[j][c][0], ui = wv * accU[j][c][1];
                    double v[16];
#pragma unroll
                    for (int c2 = 0; c2 < 8; ++c2) {
                        v[2 * c2] = c2 < NP ? ur * accW[j][c2 < NP ? c2 : 0][0] - ui * accW[j][c2 < NP ? c2 : 0][1] : 0.0;
                        v[2 * c2 + 1] = c2 < NP ? ur * accW[j][c2 < NP ? c2 : 0][1] + ui * accW[j][c2 < NP ? c2 : 0][0] : 0.0;
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {       // round 1: lanes g^1, halves of 8
                        const double snd = b0 ? v[i] : v[i + 8], kp = b0 ? v[i + 8] : v[i];
                        v[i] = kp + __shfl_xor_sync(0xffffffffu, snd, 4);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {       // round 2: lanes g^2, halves of 4
                        const double snd = b1 ? v[i] : v[i + 4], kp = b1 ? v[i + 4] : v[i];
                        v[i] = kp + __shfl_xor_sync(0xffffffffu, snd, 8);
                    }
#pragma unroll
                    for (int i = 0; i < 2; ++i) {       // round 3: lanes g^4, halves of 2
                        const double snd = b2 ? v[i] : v[i + 2], kp = b2 ? v[i + 2] : v[i];
                        v[i] = kp + __shfl_xor_sync(0xffffffffu, snd, 16);
                    }
                    sc[c].x += v[0];
                    sc[c].y += v[1];
                }
#pragma unroll
                for (int c = 0; c < NP; ++c) accU[j][c][0] = accU[j][c][1] = accW[j][c][0] = accW[j][c][1] = 0.0;
            }
        }
        // the two warps of a column tile write their slices; they are added in a fixed order when the block is written out
        {
            double2* dst = Sacc + (cw * 4 + t) * SL;
            if (c2own < NP) {
#pragma unroll
                for (int c = 0; c < NP; ++c) dst[c * NP + c2own] = sc[c];
            }
        }
        bar_sync_consumers();
        for (int i = ctid; i < 16 * NP * NP; i += 256) {
            const int wl = i / (NP * NP), e = i - wl * NP * NP, wg = wb * 16 + wl;      // walker wl of the block: column tile wl / 4, lane t = wl % 4
            const int s0 = ((wl >> 2) * 4 + (wl & 3)) * SL + e, s1 = (((wl >> 2) + 4) * 4 + (wl & 3)) * SL + e;
            const double2 x0 = Sacc[s0], x1 = Sacc[s1];
            if (wg < n_w) S[((size_t)pix * n_w + wg) * NP * NP + e] = make_double2(x0.x + x1.x, x0.y + x1.y);
        }
        bar_sync_consumers();
    }
}

// One-body intermediates of the SMW energy: H[w][x][0] = hbar_x . Theta0_x (reference x), H[w][x][1+a] = hbar_x . Theta0_{A_a}.
// grid n_w, one warp per (x, slot), lanes over p.  hbar = row n_chol of the [Lbar; hbar] operand.
__global__ void __launch_bounds__(256) k_cas_H(const double* __restrict__ hbar, const double* __restrict__ th0, const int* __restrict__ act,
                                               int n_act, double2* __restrict__ H, int N, int N_pad, int n_ref, int n_orb, int ldw0) {
    const int w = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int e = warp; e < n_orb * (1 + n_act); e += 8) {
        const int x = e / (1 + n_act), sl = e - x * (1 + n_act);
        const int c = sl == 0 ? x : act[sl - 1];
        double sr = 0.0, si = 0.0;
        if (c < n_ref) {
            const double* hx = hbar + (size_t)x * N_pad;
            const double* re = th0 + ((size_t)c * ldw0 + 2 * w) * N_pad;
            const double* im = re + N_pad;
            for (int p = lane; p < N; p += 32) {
                sr = fma(hx[p], re[p], sr);
                si = fma(hx[p], im[p], si);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { sr += __shfl_xor_sync(0xffffffffu, sr, o); si += __shfl_xor_sync(0xffffffffu, si, o); }
        }
        if (lane == 0) H[((size_t)w * n_orb + x) * CAS_HS + sl] = make_double2(sr, si);
    }
}

// Pair energies of every determinant from the S intermediates (Eq. 22 with Eq. 23 inserted): with
// Theta^d_x = s_x Theta0_x + sum_k G_d[k][x] Theta0_{h_k}  (s_x = 1 for a reference non-hole, else 0),
//   exchange  e = sum_{c in y-list} sum_{c' in x-list} coef_y[c] coef_x[c'] S[c][c'],
//   Coulomb   j = sum_{c in x-list} sum_{c' in y-list} coef_x[c] coef_y[c'] S[c][c'],
// lists = {self, the determinant's holes}.  grid (n_chunks, n_w); a chunk of ce (<= 16) pairs' S sits in shared memory, threads
// run over determinants; partial (E_K, E_J) sums per chunk are added in chunk order by k_cas_e1sum.
// With more than 6 active columns the S intermediates come in passes, one per pair of active groups (a <= b) of gs = 3
// columns: pass p(a,b) = a ng - a(a-1)/2 + (b-a) holds S on the panel list {x, y, G_a, G_b} (local index 2 + l for a column of
// G_a, 2 + gs + l for one of G_b); an entry S[c][c'] is read from the pass that contains both columns.  ng = 1 (<= 6 active
// columns, gs = 6) is the single-pass case.
template <int MAXE>     // compile-time bound of the excitation rank: the coefficient lists stay in registers
__global__ void __launch_bounds__(128) k_cas_energy(const double2* __restrict__ S, const CasPair* __restrict__ tiles, long long n_tiles,
                                                    const signed char* __restrict__ kind, const int* __restrict__ holeIdx,
                                                    const double2* __restrict__ G, double2* __restrict__ part, int n_w, int n_det, int max_exc,
                                                    int n_orb, int NP, int n_vtot, int pan_base, int gs, int ng, int npass, int ce) {
    extern __shared__ __align__(16) double2 Ss[];      // [ce pairs][npass][NP*NP]
    __shared__ int tx_s[16], ty_s[16];
    const int chunk = blockIdx.x, w = blockIdx.y, tid = threadIdx.x;
    const long long t0 = (long long)chunk * ce;
    const int nt = (int)min((long long)ce, n_tiles - t0), NP2 = NP * NP, PS = npass * NP2;
    for (int i = tid; i < nt * PS; i += 128) {
        const int tl = i / PS, r = i - tl * PS, ps = r / NP2, e = r - ps * NP2;
        Ss[i] = S[(((size_t)ps * n_tiles + (t0 + tl)) * n_w + w) * NP2 + e];
    }
    if (tid < nt) { tx_s[tid] = tiles[t0 + tid].pi - pan_base; ty_s[tid] = tiles[t0 + tid].pj - pan_base; }
    __syncthreads();
    for (int d = tid; d < n_det; d += 128) {
        const size_t v = (size_t)w * n_det + d;
        const signed char* kd = kind + (size_t)d * n_orb;
        const int* hi = holeIdx + (size_t)d * max_exc;
        int e = 0;
        while (e < max_exc && hi[e] >= 0) ++e;
        // entry 0 = self, entries 1..e = the holes: group and local index inside the group
        int grp[MAXE + 1], loc[MAXE + 1];
        grp[0] = 0; loc[0] = 0;
#pragma unroll
        for (int k = 0; k < MAXE; ++k) {
            const int ai = k < e ? hi[k] : 0;
            grp[1 + k] = ai / gs;
            loc[1 + k] = ai - grp[1 + k] * gs;
        }
        const double2* Gv = G + v * max_exc * n_orb;
        double2 ek = make_double2(0.0, 0.0), ej = make_double2(0.0, 0.0);
        for (int tl = 0; tl < nt; ++tl) {
            const int x = tx_s[tl], y = ty_s[tl];
            const int kx = kd[x], ky = kd[y];
            if (kx < 0 || ky < 0) continue;
            const double2* St = Ss + tl * PS;
            double2 cx[MAXE + 1], cy[MAXE + 1];
            cx[0] = make_double2(kx == 0 ? 1.0 : 0.0, 0.0);
            cy[0] = make_double2(ky == 0 ? 1.0 : 0.0, 0.0);
#pragma unroll
            for (int k = 0; k < MAXE; ++k) {
                const bool on = k < e;
                cx[1 + k] = on ? Gv[(size_t)k * n_orb + x] : make_double2(0.0, 0.0);
                cy[1 + k] = on ? Gv[(size_t)k * n_orb + y] : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int a = 0; a <= MAXE; ++a) {          // a: column in the y role
                if (a > e) break;
#pragma unroll
                for (int b = 0; b <= MAXE; ++b) {      // b: column in the x role
                    if (b > e) break;
                    // pass and local indices of (column a as y-role row, column b as x-role column)
                    int ga = a ? grp[a] : (b ? grp[b] : 0), gb = b ? grp[b] : ga;
                    int iy = a ? 2 + loc[a] : 1, ix = b ? 2 + loc[b] : 0;
                    if (a && b && ga != gb) {
                        if (ga < gb) ix += gs;
                        else { iy += gs; const int t2 = ga; ga = gb; gb = t2; }
                    }
                    const double2* Sp = St + (ga * ng - ga * (ga - 1) / 2 + (gb - ga)) * NP2;
                    const double2 cc = cmul(cy[a], cx[b]);
                    const double2 se = Sp[iy * NP + ix], sj = Sp[ix * NP + iy];
                    const double2 t1 = cmul(cc, se), t2 = cmul(cc, sj);
                    ek.x += t1.x; ek.y += t1.y;
                    ej.x += t2.x; ej.y += t2.y;
                }
            }
        }
        part[((size_t)chunk * n_vtot + v) * 2] = ek;
        part[((size_t)chunk * n_vtot + v) * 2 + 1] = make_double2(-2.0 * ej.x, -2.0 * ej.y);
    }
}

// Per virtual walker: E_K^d, E_J^d = chunk partials in chunk order; E1^d = 2 [sum_{x ref non-hole} H[x][self] +
// sum_k sum_x G_d[k][x] H[x][hole k]]; writes Ev[v] = {E_L, E1, E_J, E_K} for k_cas_combine.
__global__ void __launch_bounds__(128) k_cas_e1sum(const double2* __restrict__ part, int n_chunks, const double2* __restrict__ H,
                                                   const signed char* __restrict__ kind, const int* __restrict__ holeIdx,
                                                   const double2* __restrict__ G, double2* __restrict__ Ev, int n_v, int n_det, int max_exc,
                                                   int n_orb, int n_vtot) {
    const int v = blockIdx.x * 128 + threadIdx.x;
    if (v >= n_v) return;
    const int w = v / n_det, d = v - w * n_det;
    double2 ek = make_double2(0.0, 0.0), ej = make_double2(0.0, 0.0), e1 = make_double2(0.0, 0.0);
    for (int c = 0; c < n_chunks; ++c) {
        const double2 a = part[((size_t)c * n_vtot + v) * 2], b = part[((size_t)c * n_vtot + v) * 2 + 1];
        ek.x += a.x; ek.y += a.y;
        ej.x += b.x; ej.y += b.y;
    }
    const signed char* kd = kind + (size_t)d * n_orb;
    const int* hi = holeIdx + (size_t)d * max_exc;
    const double2* Hw = H + (size_t)w * n_orb * CAS_HS;
    const double2* Gv = G + (size_t)v * max_exc * n_orb;
    for (int x = 0; x < n_orb; ++x) {
        if (kd[x] < 0) continue;
        if (kd[x] == 0) { e1.x += Hw[x * CAS_HS].x; e1.y += Hw[x * CAS_HS].y; }
        for (int k = 0; k < max_exc && hi[k] >= 0; ++k) {
            const double2 t1 = cmul(Gv[(size_t)k * n_orb + x], Hw[x * CAS_HS + 1 + hi[k]]);
            e1.x += t1.x; e1.y += t1.y;
        }
    }
    e1.x *= 2.0; e1.y *= 2.0;
    Ev[4 * (size_t)v] = make_double2(e1.x + ej.x + ek.x, e1.y + ej.y + ek.y);
    Ev[4 * (size_t)v + 1] = e1;
    Ev[4 * (size_t)v + 2] = ej;
    Ev[4 * (size_t)v + 3] = ek;
}

// One warp per virtual walker v = w*n_det + d: lane 0 inverts T_d (<= 8 x 8, Gauss-Jordan with partial pivoting) and
// takes its determinant; all lanes then fill G_d.  weight = c_d det(T_d)^2 (closed shell: the same string in both spins;
// unrestricted: c_d det(T_d^alpha) from the alpha call times det(T_d^beta) from the beta call, multiplied in k_cas_combine);
// status 1 when the reference overlap or T_d is singular (that determinant is then left out of the sums).
__global__ void __launch_bounds__(128) k_cas_coef(const double2* __restrict__ T, const int* __restrict__ holes, const int* __restrict__ parts,
                                                  const double* __restrict__ coef, const int* __restrict__ st0, double2* __restrict__ G,
                                                  double2* __restrict__ wd, int* __restrict__ stv, int n_v, int n_det, int max_exc, int n_ref,
                                                  int n_virt, int n_orb, int wmode /* 0: c det^2, 1: c det (alpha), 2: det (beta) */) {
    __shared__ double2 inv_s[4][CAS_MAX_EXC][CAS_MAX_EXC];
    __shared__ int ok_s[4];
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5, v = blockIdx.x * 4 + wi;
    if (v >= n_v) return;
    const int w = v / n_det, d = v - w * n_det;
    const int* hs = holes + (size_t)d * max_exc;
    const int* ps = parts + (size_t)d * max_exc;
    int e = 0;
    while (e < max_exc && hs[e] >= 0) ++e;
    const double2* Tw = T + (size_t)w * n_virt * n_ref;
    if (lane == 0) {
        double2 M[CAS_MAX_EXC][CAS_MAX_EXC], I[CAS_MAX_EXC][CAS_MAX_EXC];
        for (int k = 0; k < e; ++k)
            for (int l = 0; l < e; ++l) {
                M[k][l] = Tw[(size_t)(ps[k] - n_ref) * n_ref + hs[l]];
                I[k][l] = make_double2(k == l ? 1.0 : 0.0, 0.0);
            }
        double2 det = make_double2(1.0, 0.0);
        bool ok = st0[w] == 0;
        for (int k = 0; k < e && ok; ++k) {
            int piv = k;
            double best = -1.0;
            for (int r = k; r < e; ++r) {
                double m = M[r][k].x * M[r][k].x + M[r][k].y * M[r][k].y;
                if (!(m == m)) m = INFINITY;
                if (m > best) { best = m; piv = r; }
            }
            if (!(best > 1e-300) || isinf(best)) { ok = false; break; }
            if (piv != k) {
                for (int c = 0; c < e; ++c) { double2 t1 = M[k][c]; M[k][c] = M[piv][c]; M[piv][c] = t1; t1 = I[k][c]; I[k][c] = I[piv][c]; I[piv][c] = t1; }
                det = make_double2(-det.x, -det.y);
            }
            det = cmul(det, M[k][k]);
            const double2 ip = crecip(M[k][k]);
            for (int c = 0; c < e; ++c) { M[k][c] = cmul(M[k][c], ip); I[k][c] = cmul(I[k][c], ip); }
            for (int r = 0; r < e; ++r) {
                if (r == k) continue;
                const double2 fct = M[r][k];
                for (int c = 0; c < e; ++c) {
                    double2 t1 = cmul(fct, M[k][c]), t2 = cmul(fct, I[k][c]);
                    M[r][c] = make_double2(M[r][c].x - t1.x, M[r][c].y - t1.y);
                    I[r][c] = make_double2(I[r][c].x - t2.x, I[r][c].y - t2.y);
                }
            }
        }
        for (int k = 0; k < e; ++k)
            for (int l = 0; l < e; ++l) inv_s[wi][k][l] = I[k][l];
        ok_s[wi] = ok ? 1 : 0;
        const double2 d2 = wmode == 0 ? cmul(det, det) : det;
        const double cf = wmode == 2 ? 1.0 : coef[d];
        wd[v] = ok ? make_double2(cf * d2.x, cf * d2.y) : make_double2(0.0, 0.0);
        stv[v] = ok ? 0 : 1;
    }
    __syncwarp();
    const bool ok = ok_s[wi] != 0;
    double2* Gv = G + (size_t)v * max_exc * n_orb;
    for (int x = lane; x < n_orb; x += 32) {
        int kind = x < n_ref ? 0 : -1;     // 0: reference non-hole, 1+m: particle p_m, -1: zero
        for (int m = 0; m < e; ++m) {
            if (hs[m] == x) kind = -1;
            if (ps[m] == x) kind = 1 + m;
        }
        for (int k = 0; k < e; ++k) {
            double2 gk = make_double2(0.0, 0.0);
            if (ok && kind == 0) {
                for (int l = 0; l < e; ++l) {
                    const double2 t1 = cmul(inv_s[wi][k][l], Tw[(size_t)(ps[l] - n_ref) * n_ref + x]);
                    gk.x -= t1.x; gk.y -= t1.y;
                }
            } else if (ok && kind > 0) {
                gk = inv_s[wi][k][kind - 1];
            }
            Gv[(size_t)k * n_orb + x] = gk;
        }
    }
}

// Theta^d panels of every virtual walker: grid (n_v, n_orb, ceil(N_pad/128)), thread = basis index p.
__global__ void __launch_bounds__(128) k_cas_theta(const double* __restrict__ th0, const double2* __restrict__ G, const int* __restrict__ holes,
                                                   double* __restrict__ thT, int N_pad, int n_ref, int n_orb, int n_det, int max_exc, int ldw0,
                                                   int ldw, int o_base) {
    const int p = blockIdx.z * 128 + threadIdx.x, x = blockIdx.y, v = blockIdx.x;
    if (p >= N_pad) return;
    const int w = v / n_det, d = v - w * n_det;
    const int* hs = holes + (size_t)d * max_exc;
    double re = 0.0, im = 0.0;
    bool is_hole = false;
    int e = 0;
    for (; e < max_exc && hs[e] >= 0; ++e) is_hole |= hs[e] == x;
    if (x < n_ref && !is_hole) {
        re = th0[((size_t)x * ldw0 + 2 * w) * N_pad + p];
        im = th0[((size_t)x * ldw0 + 2 * w + 1) * N_pad + p];
    }
    const double2* Gv = G + (size_t)v * max_exc * n_orb + x;
    for (int k = 0; k < e; ++k) {
        const double2 g = Gv[(size_t)k * n_orb];
        const double tr = th0[((size_t)hs[k] * ldw0 + 2 * w) * N_pad + p], ti = th0[((size_t)hs[k] * ldw0 + 2 * w + 1) * N_pad + p];
        re = fma(g.x, tr, fma(-g.y, ti, re));
        im = fma(g.x, ti, fma(g.y, tr, im));
    }
    thT[((size_t)(o_base + x) * ldw + 2 * v) * N_pad + p] = re;
    thT[((size_t)(o_base + x) * ldw + 2 * v + 1) * N_pad + p] = im;
}

// E = sum_d w_d E^d / sum_d w_d per real walker and energy term (Eq. 12), determinants in index order (fixed order).
__global__ void k_cas_combine(const double2* __restrict__ Ev, const double2* __restrict__ wd, const int* __restrict__ stv,
                              const int* __restrict__ st0, const double2* __restrict__ wdB, const int* __restrict__ stvB,
                              const int* __restrict__ st0B, int n_w, int n_det, double2* __restrict__ E_L, double2* __restrict__ E1,
                              double2* __restrict__ E_J, double2* __restrict__ E_K, double2* __restrict__ ovlp, int* __restrict__ st_out) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_w) return;
    double2 num[3] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0), make_double2(0.0, 0.0)}, den = make_double2(0.0, 0.0);
    for (int d = 0; d < n_det; ++d) {
        const size_t v = (size_t)w * n_det + d;
        if (stv[v] || (stvB && stvB[v])) continue;
        const double2 wv = wdB ? cmul(wd[v], wdB[v]) : wd[v];
        for (int c = 0; c < 3; ++c) {
            const double2 t1 = cmul(wv, Ev[4 * v + 1 + c]);
            num[c].x += t1.x; num[c].y += t1.y;
        }
        den.x += wv.x; den.y += wv.y;
    }
    const double m2 = den.x * den.x + den.y * den.y;
    const bool bad = st0[w] != 0 || (st0B && st0B[w] != 0) || !(m2 > 0.0) || isinf(m2);
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    double2 e[3], el = make_double2(0.0, 0.0);
    const double2 id = bad ? make_double2(nan, nan) : crecip(den);
    for (int c = 0; c < 3; ++c) {
        e[c] = bad ? make_double2(nan, nan) : cmul(num[c], id);
        el.x += e[c].x; el.y += e[c].y;
    }
    if (E_L) E_L[w] = el;
    if (E1) E1[w] = e[0];
    if (E_J) E_J[w] = e[1];
    if (E_K) E_K[w] = e[2];
    if (ovlp) ovlp[w] = bad ? make_double2(nan, nan) : den;
    if (st_out) st_out[w] = bad ? 1 : 0;
}

// ---- unrestricted SMW energy, Coulomb term by the Cholesky route (R9): for determinant d and spin s
//   X^{g,d}_s = sum_x Lbar^g_x . Theta^d_x = X0^g_s + sum_k sum_x G'_s[k][x] Z_s[A-index of hole k][g][x],
//   G'[k][x] = G_d[k][x] - [x == hole k],   Z_s[a][g][x] = Lbar^g_x . Theta0_{s, A_a}   (one DMMA GEMM per spin and call),
// and E_J^d = 1/2 sum_g (X^{g,d}_alpha + X^{g,d}_beta)^2  (R6; no opposite-spin pair blocks needed).  X0 = X0_alpha + X0_beta
// comes from the ordinary Coulomb kernel on the reference panels.  grid (determinant chunks, n_w), block 128: a thread
// holds 2, 4 or 8 Cholesky vectors of one determinant; the Z rows of 8 Cholesky vectors sit in shared memory while the
// block's determinants use them; sums over g in a fixed order.
struct XjSpin {
    const double* Z;          // [(a * ldw0 + 2w + c)][zcols]
    const double2* G;         // [n_v][max_exc][n_orb]
    const int* holes;         // [n_det][max_exc]
    const int* holeIdx;       // [n_det][max_exc]
    int n_orb, o_base, n_act;
};
constexpr int XJ_GT = 8;      // Cholesky vectors per shared-memory tile (107 KB at 6 x 70 orbitals per spin: 2 blocks per SM)
template <int GJ>             // Cholesky vectors per thread (8, 4 or 2 of the tile's 8): a block holds 128 * GJ / 8 determinants
__global__ void __launch_bounds__(128) k_cas_xj(XjSpin sa, XjSpin sb, const double* __restrict__ X0, int ldx0, int n_chol, int O_tot,
                                                long long zcols, int ldw0, int n_det, int max_exc, double2* __restrict__ EJ) {
    extern __shared__ __align__(16) double2 Zs[];      // [spin][a][Cholesky vector of the tile][x]  (x fastest: conflict-free fill)
    constexpr int TG = XJ_GT / GJ;                     // threads per determinant
    const int w = blockIdx.y, tid = threadIdx.x, j0 = (tid % TG) * GJ;
    const int d = blockIdx.x * (128 / TG) + tid / TG;  // GJ Cholesky vectors of one determinant per thread, in registers
    const bool live = d < n_det;
    const size_t v = (size_t)w * n_det + (live ? d : 0);
    const XjSpin sp[2] = {sa, sb};
    const int offB = sa.n_act * sa.n_orb * XJ_GT;
    double sr = 0.0, si = 0.0;
    for (int g0 = 0; g0 < n_chol; g0 += XJ_GT) {
        __syncthreads();
        for (int s = 0; s < 2; ++s) {
            const XjSpin& S = sp[s];
            double2* dst = Zs + (s ? offB : 0);
            const int per = S.n_orb * XJ_GT, total = S.n_act * per;
            for (int e = tid; e < total; e += 128) {
                const int a = e / per, r = e - a * per, gg = r / S.n_orb, x = r - gg * S.n_orb;
                double2 z = make_double2(0.0, 0.0);
                if (g0 + gg < n_chol) {
                    const size_t col = (size_t)(g0 + gg) * O_tot + S.o_base + x;
                    z.x = S.Z[((size_t)a * ldw0 + 2 * w) * zcols + col];
                    z.y = S.Z[((size_t)a * ldw0 + 2 * w + 1) * zcols + col];
                }
                dst[e] = z;
            }
        }
        __syncthreads();
        double xr[GJ], xi[GJ];
#pragma unroll
        for (int j = 0; j < GJ; ++j) {
            const bool on = g0 + j0 + j < n_chol;
            xr[j] = on ? X0[(size_t)(g0 + j0 + j) * ldx0 + 2 * w] : 0.0;
            xi[j] = on ? X0[(size_t)(g0 + j0 + j) * ldx0 + 2 * w + 1] : 0.0;
        }
        for (int s = 0; s < 2 && live; ++s) {
            const XjSpin& S = sp[s];
            const double2* zs = Zs + (s ? offB : 0);
            const double2* Gv = S.G + v * max_exc * S.n_orb;
            for (int k = 0; k < max_exc; ++k) {
                const int h = S.holes[(size_t)d * max_exc + k];
                if (h < 0) break;
                const double2* za = zs + ((size_t)S.holeIdx[(size_t)d * max_exc + k] * XJ_GT + j0) * S.n_orb;
                const double2* gk = Gv + (size_t)k * S.n_orb;
                for (int x0 = 0; x0 < S.n_orb; x0 += 8) {            // 8 independent loads in flight (the loop is latency bound otherwise)
                    double2 c[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) c[u] = x0 + u < S.n_orb ? __ldg(gk + x0 + u) : make_double2(0.0, 0.0);
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        if (x0 + u == h) c[u].x -= 1.0;
                        const int xx = min(x0 + u, S.n_orb - 1);
#pragma unroll
                        for (int j = 0; j < GJ; ++j) {
                            const double2 z = za[j * S.n_orb + xx];    // the same address in every thread with this hole: broadcast
                            xr[j] = fma(c[u].x, z.x, fma(-c[u].y, z.y, xr[j]));
                            xi[j] = fma(c[u].x, z.y, fma(c[u].y, z.x, xi[j]));
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < GJ; ++j) {            // rows beyond n_chol hold zeros
            sr += xr[j] * xr[j] - xi[j] * xi[j];
            si += 2.0 * xr[j] * xi[j];
        }
    }
#pragma unroll
    for (int o = 1; o < TG; o <<= 1) { sr += __shfl_xor_sync(0xffffffffu, sr, o); si += __shfl_xor_sync(0xffffffffu, si, o); }
    if (live && tid % TG == 0) EJ[v] = make_double2(0.5 * sr, 0.5 * si);
}

// Per virtual walker of an unrestricted trial: E_K^d = alpha + beta chunk partials (the factor weights carry the 1/2 per
// spin), E1^d = sum over spins of [sum_{x ref non-hole} H[x][self] + sum_k sum_x G_d[k][x] H[x][hole k]] (R6: no factor 2),
// E_J^d from k_cas_xj.
struct EsSpin {
    const double2* part; int n_chunks;
    const double2* H; const signed char* kind; const int* holeIdx; const double2* G; int n_orb;
};
__global__ void __launch_bounds__(128) k_cas_esum_u(EsSpin sa, EsSpin sb, const double2* __restrict__ EJ, double2* __restrict__ Ev, int n_v,
                                                    int n_det, int max_exc, int n_vtot) {
    const int v = blockIdx.x * 128 + threadIdx.x;
    if (v >= n_v) return;
    const int w = v / n_det, d = v - w * n_det;
    double2 ek = make_double2(0.0, 0.0), e1 = make_double2(0.0, 0.0);
    const EsSpin sp[2] = {sa, sb};
    for (int s = 0; s < 2; ++s) {
        const EsSpin& S = sp[s];
        for (int c = 0; c < S.n_chunks; ++c) {
            const double2 a = S.part[((size_t)c * n_vtot + v) * 2];
            ek.x += a.x; ek.y += a.y;
        }
        const signed char* kd = S.kind + (size_t)d * S.n_orb;
        const int* hi = S.holeIdx + (size_t)d * max_exc;
        const double2* Hw = S.H + (size_t)w * S.n_orb * CAS_HS;
        const double2* Gv = S.G + (size_t)v * max_exc * S.n_orb;
        for (int x = 0; x < S.n_orb; ++x) {
            if (kd[x] < 0) continue;
            if (kd[x] == 0) { e1.x += Hw[x * CAS_HS].x; e1.y += Hw[x * CAS_HS].y; }
            for (int k = 0; k < max_exc && hi[k] >= 0; ++k) {
                const double2 t1 = cmul(Gv[(size_t)k * S.n_orb + x], Hw[x * CAS_HS + 1 + hi[k]]);
                e1.x += t1.x; e1.y += t1.y;
            }
        }
    }
    const double2 ej = EJ[v];
    Ev[4 * (size_t)v] = make_double2(e1.x + ej.x + ek.x, e1.y + ej.y + ek.y);
    Ev[4 * (size_t)v + 1] = e1;
    Ev[4 * (size_t)v + 2] = ej;
    Ev[4 * (size_t)v + 3] = ek;
}

}  // namespace

lo_status configure_cas_kernels() {
    cudaError_t e = cudaFuncSetAttribute(k_cas_pairs<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, CpCfg<4>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_pairs<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, CpCfg<6>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_pairs<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, CpCfg<8>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_xj<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_xj<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_xj<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_cas_*): ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

// local energy with a multi-determinant trial by direct summation over determinants (Eq. 12), the
// determinants' overlaps and Green's functions by SMW updates of the reference (Eq. 20); each (walker, determinant) is a
// virtual walker of the ordinary Coulomb / exchange kernels (orbital-indexed Theta^d panels, zero where unoccupied).
lo_status launch_local_energy_cas(lo_factors* f, int n_w, const void* phi, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K,
                                  void* ovlp, int* walker_status, cudaStream_t stream) {
    CasPlan& c = *f->cas;
    const int n_orb = f->n_occ[0], n_v = n_w * c.n_det, ldw0 = 2 * c.W0cap;
    const bool smw = c.mode != 0, unres = c.has_beta;
    launch_s1(f, n_w, f->ops->dPsi[0], n_orb, c.n_ref, phi, c.dA0, c.dSt0, c.dTh0, 0, ldw0, stream);
    k_cas_T<<<n_w, 256, 0, stream>>>(f->ops->dPsi[0], n_orb, c.dTh0, (double2*)c.dT, f->N, f->N_pad, c.n_ref, c.n_virt, ldw0);
    int* stv = smw ? c.dStV : f->dStatus;
    int* stvB = smw ? c.dStVB : f->dStatus + f->Wcap;
    k_cas_coef<<<(n_v + 3) / 4, 128, 0, stream>>>((const double2*)c.dT, c.dHoles, c.dParts, c.dCoef, c.dSt0, (double2*)c.dG, (double2*)c.dWd,
                                                  stv, n_v, c.n_det, c.max_exc, c.n_ref, c.n_virt, n_orb, unres ? 1 : 0);
    if (unres) {
        // unrestricted trial: the beta strings get their own SMW data; in the direct mode their Theta^d panels follow the alpha panels
        const int n_orb_b = f->n_occ[1];
        launch_s1(f, n_w, f->ops->dPsi[1], n_orb_b, c.n_ref_b, phi_b, c.dA0B, c.dSt0B, c.dTh0B, 0, ldw0, stream);
        k_cas_T<<<n_w, 256, 0, stream>>>(f->ops->dPsi[1], n_orb_b, c.dTh0B, (double2*)c.dTB, f->N, f->N_pad, c.n_ref_b, c.n_virt_b, ldw0);
        k_cas_coef<<<(n_v + 3) / 4, 128, 0, stream>>>((const double2*)c.dTB, c.dHolesB, c.dPartsB, c.dCoef, c.dSt0B, (double2*)c.dGB,
                                                      (double2*)c.dWdB, stvB, n_v, c.n_det, c.max_exc, c.n_ref_b, c.n_virt_b, n_orb_b, 2);
        if (!smw) {
            dim3 g3b(n_v, n_orb_b, (f->N_pad + 127) / 128);
            k_cas_theta<<<g3b, 128, 0, stream>>>(c.dTh0B, (const double2*)c.dGB, c.dHolesB, f->dThT, f->N_pad, c.n_ref_b, n_orb_b, c.n_det, c.max_exc,
                                                 ldw0, f->ldw, f->o_base[1]);
        }
    }
    if (!smw) {
        dim3 g3(n_v, n_orb, (f->N_pad + 127) / 128);
        k_cas_theta<<<g3, 128, 0, stream>>>(c.dTh0, (const double2*)c.dG, c.dHoles, f->dThT, f->N_pad, c.n_ref, n_orb, c.n_det, c.max_exc, ldw0, f->ldw, 0);
        lo_status st = launch_s3_s5(f, n_v, nullptr, nullptr, nullptr, nullptr, nullptr, c.dEv, stream);
        if (st != LO_OK) return st;
    } else {
        // rearranged SMW energy (Eq. 23), per spin: S intermediates once per (tile, walker), one-body intermediates, then small
        // per-determinant forms (exchange, and for a closed-shell trial the compressed Coulomb term)
        const int WB = (n_w + 15) / 16;
        const int n_vtot = c.max_real * c.n_det;
        const double* hbar0 = f->ops->dLbar + (size_t)f->n_chol * f->O_tot * f->N_pad;
        for (int s = 0; s < (unres ? 2 : 1); ++s) {
            const int NP = s ? c.NPB : c.NP, n_act = s ? c.n_actB : c.n_act, n_orb_s = f->n_occ[s], n_ref_s = s ? c.n_ref_b : c.n_ref;
            const int pan_base = f->o_base[s];
            const long long nt = c.npair[s];               // pairs with rows (S exists once per pair)
            const CasPair* tiles = c.dPairs[s];
            const int* hidx = s ? c.dHoleIdxB : c.dHoleIdx;
            const int* actd = hidx + (size_t)c.n_det * c.max_exc;      // A_set stored behind the hole indices
            double2* S = (double2*)(s ? c.dSB : c.dS);
            double* th0 = s ? c.dTh0B : c.dTh0;
            const CUtensorMap& tm0 = s ? c.tmTh0B : c.tmTh0;
            const long long items = nt * WB;
            const int grid = (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
            // one pass per pair of active groups (a single pass for <= 6 active columns); pass p fills S[p][pair][walker]
            for (int ps = 0; ps < c.npass[s]; ++ps) {
                const int* pact = c.dPassAct[s] + (size_t)ps * 6;
                double2* Sp = S + (size_t)ps * nt * n_w * NP * NP;
                if (NP == 4)
                    k_cas_pairs<4><<<grid, 384, CpCfg<4>::SMEM, stream>>>(f->tmUf, f->tmWf, tm0, f->dWgt, f->dTiles4, tiles, items, WB, f->N_pad, ldw0, pact, Sp, n_w, pan_base);
                else if (NP == 6)
                    k_cas_pairs<6><<<grid, 384, CpCfg<6>::SMEM, stream>>>(f->tmUf, f->tmWf, tm0, f->dWgt, f->dTiles4, tiles, items, WB, f->N_pad, ldw0, pact, Sp, n_w, pan_base);
                else
                    k_cas_pairs<8><<<grid, 384, CpCfg<8>::SMEM, stream>>>(f->tmUf, f->tmWf, tm0, f->dWgt, f->dTiles4, tiles, items, WB, f->N_pad, ldw0, pact, Sp, n_w, pan_base);
            }
            k_cas_H<<<n_w, 256, 0, stream>>>(hbar0 + (size_t)pan_base * f->N_pad, th0, actd, n_act, (double2*)(s ? c.dHB : c.dH), f->N, f->N_pad,
                                             n_ref_s, n_orb_s, ldw0);
            const int ce = c.ce[s], gs = c.gs[s], ng = c.ng[s], npass = c.npass[s];
            const int n_chunks = (int)((nt + ce - 1) / ce);
            if (n_chunks > 0) {
                dim3 g4(n_chunks, n_w);
                const size_t sm4 = (size_t)ce * npass * NP * NP * 16;
                const signed char* kind = s ? c.dKindB : c.dKind;
                const double2* G = (const double2*)(s ? c.dGB : c.dG);
                double2* part = (double2*)(s ? c.dPartB : c.dPart);
                if (c.max_exc <= 2)
                    k_cas_energy<2><<<g4, 128, sm4, stream>>>(S, tiles, nt, kind, hidx, G, part, n_w, c.n_det, c.max_exc, n_orb_s, NP, n_vtot, pan_base, gs, ng, npass, ce);
                else if (c.max_exc <= 4)
                    k_cas_energy<4><<<g4, 128, sm4, stream>>>(S, tiles, nt, kind, hidx, G, part, n_w, c.n_det, c.max_exc, n_orb_s, NP, n_vtot, pan_base, gs, ng, npass, ce);
                else
                    k_cas_energy<8><<<g4, 128, sm4, stream>>>(S, tiles, nt, kind, hidx, G, part, n_w, c.n_det, c.max_exc, n_orb_s, NP, n_vtot, pan_base, gs, ng, npass, ce);
            }
        }
        if (!unres) {
            k_cas_e1sum<<<(n_v + 127) / 128, 128, 0, stream>>>((const double2*)c.dPart, c.n_chunks, (const double2*)c.dH, c.dKind, c.dHoleIdx,
                                                               (const double2*)c.dG, (double2*)c.dEv, n_v, c.n_det, c.max_exc, n_orb, n_vtot);
        } else {
            // Coulomb term by the Cholesky route (R6, R9): X0 = X0_alpha + X0_beta of the reference from the ordinary kernel on
            // the reference panels, the Z intermediates of both spins by one DMMA GEMM each, then per (walker, determinant)
            // E_J^d = 1/2 sum_g (X0^g + SMW corrections)^2  (k_cas_xj)
            const long long zcols = (long long)f->Xp * f->O_tot;
            for (int s = 0; s < 2; ++s) {
                const double* th0 = s ? c.dTh0B : c.dTh0;
                cudaMemcpy2DAsync(f->dThT + (size_t)f->o_base[s] * f->ldw * f->N_pad, (size_t)f->ldw * f->N_pad * 8, th0, (size_t)ldw0 * f->N_pad * 8,
                                  (size_t)2 * n_w * f->N_pad * 8, f->n_occ[s], cudaMemcpyDeviceToDevice, stream);
            }
            launch_coulomb_x(f, n_w, stream);
            for (int s = 0; s < 2; ++s) {
                const int n_act = s ? c.n_actB : c.n_act, na_pad = (s ? c.NPB : c.NP) - 2;
                const int* hact = s ? c.hActB : c.hAct;
                const double* th0 = s ? c.dTh0B : c.dTh0;
                for (int a = 0; a < n_act; ++a)
                    cudaMemcpyAsync(c.dThAct[s] + (size_t)a * ldw0 * f->N_pad, th0 + (size_t)hact[a] * ldw0 * f->N_pad, (size_t)ldw0 * f->N_pad * 8,
                                    cudaMemcpyDeviceToDevice, stream);
                // Z_s[(a, 2w+c)][g * O_tot + o] = Lbar^g_o . Theta0_{s, A_a}
                launch_gemm_kmajor(c.tmThAct[s], c.tmLbarRows, c.dZ[s], (long long)na_pad * ldw0, zcols, f->N_pad, zcols, f->num_sms, stream);
            }
            XjSpin xa = {c.dZ[0], (const double2*)c.dG, c.dHoles, c.dHoleIdx, f->n_occ[0], f->o_base[0], c.n_act};
            XjSpin xb = {c.dZ[1], (const double2*)c.dGB, c.dHolesB, c.dHoleIdxB, f->n_occ[1], f->o_base[1], c.n_actB};
            const size_t smx = ((size_t)std::max(c.n_act, 1) * f->n_occ[0] + (size_t)std::max(c.n_actB, 1) * f->n_occ[1]) * XJ_GT * 16;
            if (smx > 200 * 1024) { set_error("lo_local_energy_cas: active set x orbitals too large for the Coulomb intermediates in shared memory"); return LO_EINVAL; }
            // as many Cholesky vectors per thread (reuse of every G' entry) as still leaves >= 8 blocks per SM
            const long long want = 4LL * f->num_sms;
            if ((long long)n_w * ((c.n_det + 127) / 128) >= want) {
                dim3 gx((c.n_det + 127) / 128, n_w);
                k_cas_xj<8><<<gx, 128, smx, stream>>>(xa, xb, f->dXpart, f->ldw, f->n_chol, f->O_tot, zcols, ldw0, c.n_det, c.max_exc, (double2*)c.dEJu);
            } else if ((long long)n_w * ((c.n_det + 63) / 64) >= want) {
                dim3 gx((c.n_det + 63) / 64, n_w);
                k_cas_xj<4><<<gx, 128, smx, stream>>>(xa, xb, f->dXpart, f->ldw, f->n_chol, f->O_tot, zcols, ldw0, c.n_det, c.max_exc, (double2*)c.dEJu);
            } else {
                dim3 gx((c.n_det + 31) / 32, n_w);
                k_cas_xj<2><<<gx, 128, smx, stream>>>(xa, xb, f->dXpart, f->ldw, f->n_chol, f->O_tot, zcols, ldw0, c.n_det, c.max_exc, (double2*)c.dEJu);
            }
            EsSpin ea = {(const double2*)c.dPart, c.n_chunks, (const double2*)c.dH, c.dKind, c.dHoleIdx, (const double2*)c.dG, f->n_occ[0]};
            EsSpin eb = {(const double2*)c.dPartB, c.n_chunksB, (const double2*)c.dHB, c.dKindB, c.dHoleIdxB, (const double2*)c.dGB, f->n_occ[1]};
            k_cas_esum_u<<<(n_v + 127) / 128, 128, 0, stream>>>(ea, eb, (const double2*)c.dEJu, (double2*)c.dEv, n_v, c.n_det, c.max_exc, n_vtot);
        }
    }
    k_cas_combine<<<(n_w + 127) / 128, 128, 0, stream>>>((const double2*)c.dEv, (const double2*)c.dWd, stv, c.dSt0,
                                                         unres ? (const double2*)c.dWdB : nullptr, unres ? stvB : nullptr,
                                                         unres ? c.dSt0B : nullptr, n_w, c.n_det,
                                                         (double2*)E_L, (double2*)E1, (double2*)E_J, (double2*)E_K, (double2*)ovlp, walker_status);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("lo_local_energy_cas: kernel launch failed: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

}  // namespace lo
