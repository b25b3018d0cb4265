// lo_kernels.cu -- the hot path of lo_local_energy (steps S1-S5 of SURVEY.md 8(a)), hand-written for sm_100a.
//
//   k_overlap   A_w = Psi^T Phi_w   real x complex GEMM on the DMMA pipe
//   k_inverse   A_w^-1 by in-place Gauss-Jordan with partial pivoting, in shared memory (global fallback for big O);
//               k_inverse_reg: register-resident variant for O <= 48
//   k_theta     Theta_w = Phi_w A_w^-1 (Eq. 15) as one real GEMM on the DMMA pipe, written as Theta^T panels
//               [o][2w+c][p]
//   k_coulomb   X = [Lbar; hbar] . Theta   real FP64 GEMM on the DMMA pipe, split-K partials  (Eq. 16 Coulomb part);
//               also the propagator GEMM B = Lt . x (NEXT-1, with k_pack_x)
//   k_ej        X = sum of partials, E_J partial sums of X^2 (complex square), E1 from the hbar row
//   k_exchange  grouped variable-rank dual GEMM a = U Theta_j, b = W Theta_i with fused weight * a * b reduction
//               (Eq. 19/22 exchange part); <true>: also the compressed Coulomb projections (NEXT-3)
//   k_finalize  E_K = sum of CTA partials, E_L = E1 + E_J + E_K, NaN for singular walkers
//   (the multi-determinant kernels k_cas_* are in lo_cas.cu; the shared device helpers in lo_device.cuh)
//
// FP64 on sm_100a has no tcgen05 path; the FP64 tensor instruction is the warp-level DMMA.8x8x4
// (mma.sync.aligned.m8n8k4.f64), measured at 37.1 TFLOP/s on this B200 (same rate as the DFMA pipe, but one
// instruction carries 256 FMAs, so fragments can be fed from shared memory at 25% of its bandwidth).
// Fragment layout (PTX ISA, m8n8k4 f64): lane = 4*g + t;  A: (row g, k t);  B: (k t, col g);  C: (row g, cols 2t, 2t+1).
// Both operands are K-major; TMA (cp.async.bulk.tensor, 128-byte swizzle) stages [rows][16 doubles] tiles into shared
// memory behind mbarriers, and a fixed permutation of k inside the K tile makes the 64-bit fragment loads of a
// half-warp hit 16 distinct 8-byte banks (see frag_off).
#include <cuda.h>

#include <cstdio>

#include "lo_internal.h"

#include "lo_device.cuh"

namespace lo {

namespace {

// ------------------------------------------------------------------------------------------------ S1: overlap
// A_w[i][j] = sum_p Psi[p][i] Phi_w[p][j]  as a real GEMM on the DMMA pipe: M = i (block of 32 per CTA), N = (j, re/im)
// = the 2*O interleaved doubles of a Phi row, K = p.  grid (row blocks of MFB fragments, n_w, column blocks), 8 warps;
// warp w owns column fragments w, w+8, ... (NFW of them) and all MFB row fragments.  Psi / Phi rows are staged OV_PC at a time through shared memory;
// both operands are stored with k (= p) as the slow index, so a fragment load reads 8 consecutive doubles of 4 rows and
// a leading dimension = 4 (mod 16) doubles keeps the 16 lanes of a half-warp on distinct 8-byte banks.
constexpr int OV_PC = 32;
constexpr int OV_LDA = 52;   // >= 5 row fragments (40 columns), = 4 (mod 16)
constexpr int OV_NFB = 40;   // column fragments per CTA (grid.z blocks of 320 real columns = 160 orbitals): two staging buffers stay < 200 KB
__host__ __device__ inline int ov_ldb(int O) { int nf8 = min((2 * O + 7) / 8, OV_NFB) * 8; return nf8 + ((4 - nf8 % 16) + 16) % 16; }

template <int MFB, int NFW>
__global__ void __launch_bounds__(256) k_overlap(const double* __restrict__ psi, const double2* __restrict__ phi, double2* __restrict__ A,
                                                 int N, int O, int ldpsi) {
    extern __shared__ __align__(16) double sm[];
    const int LDB = ov_ldb(O), nf0 = blockIdx.z * OV_NFB, NF = min((2 * O + 7) / 8 - nf0, OV_NFB), c0 = nf0 * 8;
    const int buf_doubles = OV_PC * (OV_LDA + LDB);     // two buffers: [OV_PC][OV_LDA] Psi rows, [OV_PC][LDB] Phi rows
    const int i0 = blockIdx.x * (MFB * 8), w = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    const double* phw = reinterpret_cast<const double*>(phi + (size_t)w * N * O);
    const int O2 = 2 * O, ncb = NF * 8;
    double acc[MFB][NFW][2];
#pragma unroll
    for (int a = 0; a < MFB; ++a)
#pragma unroll
        for (int b = 0; b < NFW; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    // asynchronous staging (cp.async, zero fill outside the matrix): chunk k+1 is in flight while chunk k feeds the MMAs
    auto issue = [&](int p0, double* As, double* Bs) {
        for (int e = tid; e < OV_PC * (MFB * 8); e += 256) {
            const int pp = e / (MFB * 8), c = e - pp * (MFB * 8), pg = p0 + pp;
            const bool ok = pg < N && i0 + c < O;
            cp_async8(As + pp * OV_LDA + c, ok ? psi + (size_t)pg * ldpsi + i0 + c : psi, ok);
        }
        for (int e = tid; e < OV_PC * (ncb / 2); e += 256) {
            const int pp = e / (ncb / 2), c = 2 * (e - pp * (ncb / 2)), pg = p0 + pp;
            const bool ok = pg < N && c0 + c < O2;
            cp_async16(Bs + pp * LDB + c, ok ? phw + (size_t)pg * O2 + c0 + c : phw, ok);
        }
        cp_async_commit();
    };
    issue(0, sm, sm + OV_PC * OV_LDA);
    int kbuf = 0;
    for (int p0 = 0; p0 < N; p0 += OV_PC, kbuf ^= 1) {
        const double* As = sm + kbuf * buf_doubles;
        const double* Bs = As + OV_PC * OV_LDA;
        if (p0 + OV_PC < N) {
            double* nb = sm + (kbuf ^ 1) * buf_doubles;
            issue(p0 + OV_PC, nb, nb + OV_PC * OV_LDA);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
#pragma unroll
        for (int ks = 0; ks < OV_PC / 4; ++ks) {
            double a[MFB], b[NFW];
#pragma unroll
            for (int mf = 0; mf < MFB; ++mf) a[mf] = As[(ks * 4 + t) * OV_LDA + mf * 8 + g];
#pragma unroll
            for (int j = 0; j < NFW; ++j) {
                const int nf = min(warp + 8 * j, NF - 1);
                b[j] = Bs[(ks * 4 + t) * LDB + nf * 8 + g];
            }
#pragma unroll
            for (int mf = 0; mf < MFB; ++mf)
#pragma unroll
                for (int j = 0; j < NFW; ++j) mma884(acc[mf][j][0], acc[mf][j][1], a[mf], b[j]);
        }
        __syncthreads();      // the buffer is refilled by the issue of the next iteration
    }
#pragma unroll
    for (int mf = 0; mf < MFB; ++mf)
#pragma unroll
        for (int j = 0; j < NFW; ++j) {
            const int nf = warp + 8 * j, i = i0 + mf * 8 + g, jo = (nf0 + nf) * 4 + t;
            if (nf < NF && i < O && jo < O) A[((size_t)w * O + i) * O + jo] = make_double2(acc[mf][j][0], acc[mf][j][1]);
        }
}

// ------------------------------------------------------------------------------------------------ S1: inverse
// In-place Gauss-Jordan inversion with partial (row) pivoting.  One CTA per walker; the O x O complex matrix
// lives in shared memory (IN_SMEM) or is updated in place in the global workspace (L2 resident) when it does
// not fit.  status[w] = 1 and A^-1 = NaN when a pivot is zero / non-finite.
// Step k (3 barriers): (1) warp 0 finds the pivot of column k among rows k..O-1 (largest |.|^2, lowest row on ties) and
// publishes the row, the pivot value and the singular flag; (2) rows k and piv are exchanged while the new row k is
// scaled by 1/pivot (copy kept in rowk), column k is saved in colk -- nobody writes column k in this phase; (3) every
// other row r gets M[r][c] -= colk[r] * rowk[c], and column k becomes -colk[r]/pivot (1/pivot on the diagonal).
// Threads form a 16 x 16 grid over (row, column) so that the update reads each rowk / colk entry once per thread.
constexpr int INV_CT = 9;   // register-cached rowk entries per thread: covers O <= 144
template <bool IN_SMEM>
__global__ void __launch_bounds__(256) k_inverse(double2* __restrict__ Aws, int* __restrict__ status, int O) {
    extern __shared__ __align__(16) double sm[];
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, tx = tid & 15, ty = tid >> 4;
    double2* Ag = Aws + (size_t)w * O * O;
    double2* colk = reinterpret_cast<double2*>(sm);              // [O]
    double2* rowk = colk + O;                                    // [O]
    double2* pvs = rowk + O;                                     // [1] pivot value
    int* perm = reinterpret_cast<int*>(pvs + 1);                 // [O] padded to a multiple of 4
    int* ctl = perm + ((O + 3) & ~3);                            // [0] pivot row, [1] singular flag (+2 pad)
    double2* M = IN_SMEM ? reinterpret_cast<double2*>(ctl + 4) : Ag;
    const int OO = O * O;
    if (IN_SMEM) {
        for (int e = tid; e < OO; e += 256) M[e] = Ag[e];
    }
    if (tid == 0) ctl[1] = 0;
    __syncthreads();
    const bool cached = O <= 16 * INV_CT;
    for (int k = 0; k < O; ++k) {
        if (warp == 0) {
            double best = -1.0;
            int bi = k;
            for (int r = k + lane; r < O; r += 32) {
                double2 v = M[r * O + k];
                double m = v.x * v.x + v.y * v.y;
                if (!(m == m)) m = INFINITY;   // NaN -> treated as non-finite pivot
                if (m > best) { best = m; bi = r; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                double ob = __shfl_xor_sync(0xffffffffu, best, o);
                int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
            }
            if (lane == 0) {
                ctl[0] = bi;
                perm[k] = bi;
                pvs[0] = M[bi * O + k];
                if (!(best > 1e-300) || isinf(best)) ctl[1] = 1;
            }
        }
        __syncthreads();
        if (ctl[1]) break;   // uniform
        const int piv = ctl[0];
        const double2 inv = crecip(pvs[0]);
        for (int c = tid; c < O; c += 256) {
            // column k of the exchanged matrix (read only here), then rows k / piv without their column-k entries
            colk[c] = M[(c == k ? piv : (c == piv ? k : c)) * O + k];
            if (c != k) {
                const double2 a = M[piv * O + c], b = M[k * O + c];
                const double2 ak = cmul(a, inv);
                rowk[c] = ak;
                M[k * O + c] = ak;
                if (piv != k) M[piv * O + c] = b;
            }
        }
        __syncthreads();
        if (cached) {
            double2 v[INV_CT];
#pragma unroll
            for (int b = 0; b < INV_CT; ++b) { const int c = tx + 16 * b; v[b] = (c < O && c != k) ? rowk[c] : make_double2(0.0, 0.0); }
            for (int r = ty; r < O; r += 16) {
                if (r == k) continue;
                const double2 f = colk[r];
                double2* Mr = M + r * O;
#pragma unroll
                for (int b = 0; b < INV_CT; ++b) {
                    const int c = tx + 16 * b;
                    if (c < O && c != k) {
                        double2 m = Mr[c];
                        m.x = fma(-f.x, v[b].x, fma(f.y, v[b].y, m.x));
                        m.y = fma(-f.x, v[b].y, fma(-f.y, v[b].x, m.y));
                        Mr[c] = m;
                    }
                }
            }
        } else {
            for (int r = ty; r < O; r += 16) {
                if (r == k) continue;
                const double2 f = colk[r];
                double2* Mr = M + r * O;
                for (int c = tx; c < O; c += 16) {
                    if (c == k) continue;
                    const double2 vv = rowk[c];
                    double2 m = Mr[c];
                    m.x = fma(-f.x, vv.x, fma(f.y, vv.y, m.x));
                    m.y = fma(-f.x, vv.y, fma(-f.y, vv.x, m.y));
                    Mr[c] = m;
                }
            }
        }
        for (int r = tid; r < O; r += 256) {
            const double2 f = colk[r];
            M[r * O + k] = (r == k) ? inv : make_double2(-(f.x * inv.x - f.y * inv.y), -(f.x * inv.y + f.y * inv.x));
        }
        __syncthreads();
    }
    const bool singular = ctl[1] != 0;
    if (!singular) {
        // undo the row interchanges: A^-1 = (P A)^-1 P, i.e. swap columns in reverse order
        for (int k = O - 1; k >= 0; --k) {
            int piv = perm[k];
            if (piv != k) {
                for (int r = tid; r < O; r += 256) {
                    double2 a = M[r * O + k], b = M[r * O + piv];
                    M[r * O + k] = b;
                    M[r * O + piv] = a;
                }
                __syncthreads();
            }
        }
    }
    __syncthreads();
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    if (singular) {
        for (int e = tid; e < OO; e += 256) Ag[e] = make_double2(nan, nan);
    } else if (IN_SMEM) {
        for (int e = tid; e < OO; e += 256) Ag[e] = M[e];
    }
    if (tid == 0) status[w] = singular ? 1 : 0;
}

// Register-resident variant for O <= 16*RT <= 48: the 16 x 16 thread grid keeps the matrix in registers (thread (tx,ty) owns
// rows ty + 16a, columns tx + 16b); only the pivot column and the two exchanged rows go through (double-buffered) shared
// memory, so a step costs 3 barriers and no shared-memory traffic for the rank-1 update.  Same pivoting rule and the
// same column un-permutation as k_inverse.
template <int RT>
__global__ void __launch_bounds__(256) k_inverse_reg(double2* __restrict__ Aws, int* __restrict__ status, int O) {
    __shared__ double2 colbuf[2][RT * 16], rowk[2][RT * 16], rowp[2][RT * 16], pvs;
    __shared__ int perm[RT * 16], dest[RT * 16], ctl[2];
    const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, tx = tid & 15, ty = tid >> 4;
    double2* Ag = Aws + (size_t)w * O * O;
    double2 M[RT][RT];
#pragma unroll
    for (int a = 0; a < RT; ++a)
#pragma unroll
        for (int b = 0; b < RT; ++b) {
            const int r = ty + 16 * a, c = tx + 16 * b;
            M[a][b] = (r < O && c < O) ? Ag[(size_t)r * O + c] : make_double2(0.0, 0.0);
        }
    if (tid == 0) ctl[1] = 0;
    __syncthreads();
    for (int k = 0; k < O; ++k) {
        const int kb = k >> 4, kx = k & 15, ka = kb, ky = kx, buf = k & 1;
        if (tx == kx) {
#pragma unroll
            for (int a = 0; a < RT; ++a)
#pragma unroll
                for (int b = 0; b < RT; ++b)
                    if (b == kb) colbuf[buf][ty + 16 * a] = M[a][b];
        }
        __syncthreads();
        if (warp == 0) {
            double best = -1.0;
            int bi = k;
            for (int r = k + lane; r < O; r += 32) {
                const double2 v = colbuf[buf][r];
                double m = v.x * v.x + v.y * v.y;
                if (!(m == m)) m = INFINITY;
                if (m > best) { best = m; bi = r; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double ob = __shfl_xor_sync(0xffffffffu, best, o);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
            }
            if (lane == 0) {
                ctl[0] = bi;
                perm[k] = bi;
                pvs = colbuf[buf][bi];
                if (!(best > 1e-300) || isinf(best)) ctl[1] = 1;
            }
        }
        __syncthreads();
        if (ctl[1]) break;   // uniform
        const int piv = ctl[0], pa = piv >> 4, py = piv & 15;
        const double2 inv = crecip(pvs);
#pragma unroll
        for (int a = 0; a < RT; ++a) {
            if (ty == ky && a == ka) {
#pragma unroll
                for (int b = 0; b < RT; ++b) rowk[buf][tx + 16 * b] = M[a][b];
            }
            if (ty == py && a == pa) {
#pragma unroll
                for (int b = 0; b < RT; ++b) rowp[buf][tx + 16 * b] = M[a][b];
            }
        }
        __syncthreads();
        double2 v[RT];
#pragma unroll
        for (int b = 0; b < RT; ++b) v[b] = cmul(rowp[buf][tx + 16 * b], inv);
#pragma unroll
        for (int a = 0; a < RT; ++a) {
            const int r = ty + 16 * a;
            const bool is_k = r == k, is_p = r == piv && piv != k;
            const double2 f = is_p ? colbuf[buf][k] : colbuf[buf][r];
#pragma unroll
            for (int b = 0; b < RT; ++b) {
                const int c = tx + 16 * b;
                if (is_k) {
                    M[a][b] = c == k ? inv : v[b];
                } else {
                    const double2 base = is_p ? rowk[buf][c] : M[a][b];
                    double2 m;
                    if (c == k) {
                        m = make_double2(-(f.x * inv.x - f.y * inv.y), -(f.x * inv.y + f.y * inv.x));
                    } else {
                        m.x = fma(-f.x, v[b].x, fma(f.y, v[b].y, base.x));
                        m.y = fma(-f.x, v[b].y, fma(-f.y, v[b].x, base.y));
                    }
                    M[a][b] = m;
                }
            }
        }
    }
    __syncthreads();
    const bool singular = ctl[1] != 0;
    if (tid == 0 && !singular) {
        // column un-permutation A^-1 = (P A)^-1 P: the swaps of k_inverse applied to an index list, then inverted
        for (int c = 0; c < O; ++c) dest[c] = c;            // dest used as position -> content first
        for (int k = O - 1; k >= 0; --k) {
            const int p2 = perm[k];
            const int t1 = dest[k]; dest[k] = dest[p2]; dest[p2] = t1;
        }
        for (int j = 0; j < O; ++j) perm[dest[j]] = j;      // perm reused as content -> position
    }
    __syncthreads();
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int a = 0; a < RT; ++a)
#pragma unroll
        for (int b = 0; b < RT; ++b) {
            const int r = ty + 16 * a, c = tx + 16 * b;
            if (r < O && c < O) {
                if (singular) Ag[(size_t)r * O + c] = make_double2(nan, nan);
                else Ag[(size_t)r * O + perm[c]] = M[a][b];
            }
        }
    if (tid == 0) status[w] = singular ? 1 : 0;
}

// ------------------------------------------------------------------------------------------------ S1: Theta
// Theta[p][i] = sum_j Phi[p][j] Ainv[j][i] (complex x complex, Eq. 15) as ONE real GEMM on the DMMA pipe, computed
// transposed so that the output fragments land in the Theta^T panel layout [o][2w+c'][p]:
//   ThT[(i,c')][p] = sum_{(j,c)} Bt[(i,c')][(j,c)] * Phi[p][(j,c)],   Bt[(i,0)][(j,0)] = Re Ainv[j][i], Bt[(i,0)][(j,1)] = -Im,
//                                                                     Bt[(i,1)][(j,0)] = Im,            Bt[(i,1)][(j,1)] = Re.
// M = (i,c') (block of MFB fragments of 8 rows per CTA), N = p (64 per CTA, 8 per warp), K = (j,c) = the 2*O interleaved
// doubles of a Phi row.  grid (N_pad/64 rounded up, M blocks, n_w).  K is staged TH_KC doubles at a time; both smem
// operands are K-major with leading dimension TH_KC + 4 (= 4 mod 16: conflict-free fragment loads).  Rows p in
// [N, N_pad) are written as zeros.
constexpr int TH_KC = 32;
constexpr int TH_LD = TH_KC + 4;

template <int MFB>
__global__ void __launch_bounds__(256) k_theta(const double2* __restrict__ phi, const double2* __restrict__ Ainv, double* __restrict__ thT,
                                               int N, int N_pad, int O, int o_base, int ldw) {
    extern __shared__ __align__(16) double sm[];
    constexpr int BUF = (MFB * 8 + 64) * TH_LD;      // per buffer: Bt [MFB*8][TH_LD] then Ph [64][TH_LD]; two buffers
    constexpr int NREG = (MFB * 4 * (TH_KC / 2) + 255) / 256;
    const int p0 = blockIdx.x * 64, m0 = blockIdx.y * MFB * 8, w = blockIdx.z;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    const int O2 = 2 * O, ib0 = m0 / 2, ni = MFB * 4;
    const double* phw = reinterpret_cast<const double*>(phi + (size_t)w * N * O);
    const double2* Aw = Ainv + (size_t)w * O * O;
    double acc[MFB][2];
#pragma unroll
    for (int a = 0; a < MFB; ++a) acc[a][0] = acc[a][1] = 0.0;
    // Pipeline over the K chunks: the Phi rows of chunk k+1 arrive by cp.async and the A^-1 entries of chunk k+1 sit in
    // registers (loads in flight) while the MMAs of chunk k run; they are expanded into the 2x2 real blocks of Bt afterwards.
    auto issue_phi = [&](int k0, double* Ph) {
        for (int e = tid; e < 64 * (TH_KC / 2); e += 256) {
            const int pp = e / (TH_KC / 2), k = 2 * (e - pp * (TH_KC / 2)), pg = p0 + pp, kk = k0 + k;
            const bool ok = pg < N && kk < O2;
            cp_async16(Ph + pp * TH_LD + k, ok ? phw + (size_t)pg * O2 + kk : phw, ok);
        }
        cp_async_commit();
    };
    auto load_ainv = [&](int k0, double2 (&v)[NREG]) {
#pragma unroll
        for (int r = 0; r < NREG; ++r) {
            // consecutive threads take consecutive j of one i: their 128-bit stores below fill one Bt row contiguously
            const int e = tid + 256 * r, ii = e / (TH_KC / 2), jj = e - ii * (TH_KC / 2), i = ib0 + ii, j = k0 / 2 + jj;
            v[r] = (e < (TH_KC / 2) * ni && i < O && j < O) ? Aw[(size_t)j * O + i] : make_double2(0.0, 0.0);
        }
    };
    auto store_bt = [&](double* Bt, const double2 (&v)[NREG]) {
#pragma unroll
        for (int r = 0; r < NREG; ++r) {
            const int e = tid + 256 * r, ii = e / (TH_KC / 2), jj = e - ii * (TH_KC / 2);
            if (e < (TH_KC / 2) * ni) {
                double* r0 = Bt + (2 * ii) * TH_LD + 2 * jj;
                *reinterpret_cast<double2*>(r0) = make_double2(v[r].x, -v[r].y);
                *reinterpret_cast<double2*>(r0 + TH_LD) = make_double2(v[r].y, v[r].x);
            }
        }
    };
    double2 av[NREG];
    issue_phi(0, sm + MFB * 8 * TH_LD);
    load_ainv(0, av);
    store_bt(sm, av);
    cp_async_wait<0>();
    __syncthreads();
    int kbuf = 0;
    for (int k0 = 0; k0 < O2; k0 += TH_KC, kbuf ^= 1) {
        const double* Bt = sm + kbuf * BUF;
        const double* Ph = Bt + MFB * 8 * TH_LD;
        double* nBt = sm + (kbuf ^ 1) * BUF;
        const bool more = k0 + TH_KC < O2;
        if (more) {
            issue_phi(k0 + TH_KC, nBt + MFB * 8 * TH_LD);
            load_ainv(k0 + TH_KC, av);
        }
        const int nks = min(TH_KC / 4, (O2 - k0 + 3) / 4);      // K tail: whole k-steps of zeros are skipped (uniform)
#pragma unroll
        for (int ks = 0; ks < TH_KC / 4; ++ks) {
            if (ks >= nks) break;
            const double b = Ph[(warp * 8 + g) * TH_LD + ks * 4 + t];
            double a[MFB];
#pragma unroll
            for (int mf = 0; mf < MFB; ++mf) a[mf] = Bt[(mf * 8 + g) * TH_LD + ks * 4 + t];
#pragma unroll
            for (int mf = 0; mf < MFB; ++mf) mma884(acc[mf][0], acc[mf][1], a[mf], b);
        }
        if (more) {
            store_bt(nBt, av);
            cp_async_wait<0>();
        }
        __syncthreads();
    }
    const int p = p0 + warp * 8 + 2 * t;
    if (p < N_pad) {
#pragma unroll
        for (int mf = 0; mf < MFB; ++mf) {
            const int m = m0 + mf * 8 + g, i = m >> 1, c = m & 1;
            if (i < O)
                *reinterpret_cast<double2*>(thT + ((size_t)(o_base + i) * ldw + 2 * w + c) * N_pad + p) = make_double2(acc[mf][0], acc[mf][1]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ S3: Coulomb GEMM
// X[g][c] = sum_{o,p} LbarD[g][o][p] thT[o][c][p]; CTA tile 128 x 128, K tile 16, 8 warps of 64 x 32, 4-stage
// TMA/mbarrier pipeline that runs across work items.  Work item = (row block, column block, K split); the K range
// (flattened over (o, p-tile)) is cut into `nsplit` nearly equal parts to fill 148 SMs; partials go to Xpart[split].
constexpr int CO_STAGES = 4;
constexpr int CO_STAGE_BYTES = (CO_BM + 128) * 128;
constexpr int CO_SMEM = CO_STAGES * CO_STAGE_BYTES + 1024 + 128;

struct CoItem {
    int rb, nb, sp, ks0, nsteps;
};
__device__ __forceinline__ CoItem co_item(long long q, int RB, int NB, int nsplit, int ksteps) {
    CoItem it;
    it.nb = (int)(q % NB);
    long long r = q / NB;
    it.rb = (int)(r % RB);
    it.sp = (int)(r / RB);
    int base = ksteps / nsplit, rem = ksteps % nsplit;
    it.ks0 = it.sp * base + min(it.sp, rem);
    it.nsteps = base + (it.sp < rem ? 1 : 0);
    return it;
}

// RAGGED (the batch is not a multiple of 64 walkers): the warps are numbered column-slice first (the two warps of a
// 32-column slice sit on different schedulers) and a warp whose slice holds no walker issues no MMAs.
// NWN = column slices of 32 real columns (16 walkers) the 8 consumer warps are spread over: 4 for whole 64-walker blocks
// (warp tile 64 x 32), 2 / 1 for batches of <= 32 / <= 16 walkers (warp tiles 32 x 32 / 16 x 32: all warps keep working and
// only the Theta rows that exist are staged, through the 32-row tensor map tmT32) -- the paper's batch of 16 walkers per
// GPU ran on 2 of 8 warps before.
template <bool RAGGED, int NWN>
__global__ void __launch_bounds__(384, 1) k_coulomb(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmT,
                                                    const __grid_constant__ CUtensorMap tmT32, double* __restrict__ Xpart, int Xp, int O_tot,
                                                    int N_pad, int ldw, int RB, int NB, int nsplit, int n_cols) {
    constexpr int MF = 2 * NWN;                       // row fragments per warp
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full = sbase + CO_STAGES * CO_STAGE_BYTES, empty = full + 8 * CO_STAGES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KT = N_pad / KTILE, ksteps = O_tot * KT;
    const long long n_items = (long long)RB * NB * nsplit;
    if (tid == 0) {
        prefetch_tmap(&tmA);
        prefetch_tmap(&tmT);
        for (int i = 0; i < CO_STAGES; ++i) { mbar_init(full + 8 * i, 1); mbar_init(empty + 8 * i, 8); }
        fence_barrier_init();
    }
    __syncthreads();
    if (warp < 4) {
        // ===== producer warpgroup; one lane drives TMA, running ahead of the consumers by up to CO_STAGES stages
        reg_dec_producer();
        if (warp == 0 && lane == 0) {
            int slot = 0;
            uint32_t phase = 0;
            for (long long q = blockIdx.x; q < n_items; q += gridDim.x) {
                const CoItem it = co_item(q, RB, NB, nsplit, ksteps);
                for (int s = 0; s < it.nsteps; ++s) {
                    const int ks = it.ks0 + s;
                    const int o = ks / KT, kt = ks - o * KT;
                    mbar_wait(empty + 8 * slot, phase ^ 1);
                    const uint32_t st = sbase + slot * CO_STAGE_BYTES, bar = full + 8 * slot;
                    mbar_expect_tx(bar, NWN == 4 ? CO_STAGE_BYTES : (CO_BM + 32 * NWN) * 128);
                    tma_load_2d(st, &tmA, o * N_pad + kt * KTILE, it.rb * CO_BM, bar);
                    if constexpr (NWN == 4) tma_load_2d(st + CO_BM * 128, &tmT, kt * KTILE, o * ldw + it.nb * 128, bar);
                    else
                        for (int j = 0; j < NWN; ++j) tma_load_2d(st + (CO_BM + 32 * j) * 128, &tmT32, kt * KTILE, o * ldw + it.nb * 128 + 32 * j, bar);
                    if (++slot == CO_STAGES) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }
    // ===== 8 consumer warps (8 MF x 32 each)
    reg_inc_consumer();
    const int cw = warp - 4, g = lane >> 2, t = lane & 3;
    const int wm = NWN == 4 ? (RAGGED ? (cw & 1) : (cw >> 2)) : cw / NWN, wn = NWN == 4 ? (RAGGED ? (cw >> 1) : (cw & 3)) : cw % NWN;
    double acc[MF][4][2];
#pragma unroll
    for (int a = 0; a < MF; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t a_row = (uint32_t)(wm * MF * 8 + g) * 128, b_row = (uint32_t)(CO_BM + wn * 32 + g) * 128;
    int cslot = 0;
    uint32_t cphase = 0;
    for (long long q = blockIdx.x; q < n_items; q += gridDim.x) {
        const CoItem it = co_item(q, RB, NB, nsplit, ksteps);
        if (RAGGED && NWN == 4 && it.nb * 128 + wn * 32 >= n_cols) {          // warp-uniform: no walker in this warp's 32 columns
            for (int s = 0; s < it.nsteps; ++s) {
                mbar_wait(full + 8 * cslot, cphase);
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + 8 * cslot);
                if (++cslot == CO_STAGES) { cslot = 0; cphase ^= 1; }
            }
            continue;
        }
        for (int s = 0; s < it.nsteps; ++s) {
            mbar_wait(full + 8 * cslot, cphase);
            const uint32_t st = sbase + cslot * CO_STAGE_BYTES;
#pragma unroll
            for (int ks = 0; ks < KTILE / 4; ++ks) {
                double a[MF], b[4];
#pragma unroll
                for (int mf = 0; mf < MF; ++mf) a[mf] = lds_f64(st + a_row + mf * 1024 + xo[ks]);
#pragma unroll
                for (int nf = 0; nf < 4; ++nf) b[nf] = lds_f64(st + b_row + nf * 1024 + xo[ks]);
                if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                for (int mf = 0; mf < MF; ++mf)
#pragma unroll
                    for (int nf = 0; nf < 4; ++nf) mma884(acc[mf][nf][0], acc[mf][nf][1], a[mf], b[nf]);
            }
            if (++cslot == CO_STAGES) { cslot = 0; cphase ^= 1; }
        }
        double* Xs = Xpart + (size_t)it.sp * Xp * ldw;
#pragma unroll
        for (int mf = 0; mf < MF; ++mf)
#pragma unroll
            for (int nf = 0; nf < 4; ++nf) {
                int row = it.rb * CO_BM + wm * MF * 8 + mf * 8 + g;
                int col = it.nb * 128 + wn * 32 + nf * 8 + 2 * t;
                *reinterpret_cast<double2*>(Xs + (size_t)row * ldw + col) = make_double2(acc[mf][nf][0], acc[mf][nf][1]);
                acc[mf][nf][0] = acc[mf][nf][1] = 0.0;
            }
    }
}

// X = sum over K-split partials (written back to partial 0, the buffer lo_coulomb_x exposes); E_J partial sums per
// 128-row chunk: sum_g (X^g)^2 (complex square), the hbar row (g == n_chol) gives E1.  Fixed-order
// reductions.  grid (Wcap/32, Xp/128), block 256: lane = walker, warp = row stride.
__global__ void __launch_bounds__(256) k_ej(double* __restrict__ Xpart, double2* __restrict__ EJpart, double2* __restrict__ E1raw, int Xp,
                                            int ldw, int nsplit, int n_chol, int Wcap) {
    __shared__ double2 red[8][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int w = blockIdx.x * 32 + lane, chunk = blockIdx.y;
    double2 s = make_double2(0.0, 0.0);
    for (int rr = warp; rr < 128; rr += 8) {
        int row = chunk * 128 + rr;
        double2* x0 = reinterpret_cast<double2*>(Xpart + (size_t)row * ldw) + w;
        double2 x = *x0;
        for (int sp = 1; sp < nsplit; ++sp) {
            double2 y = *(reinterpret_cast<const double2*>(Xpart + ((size_t)sp * Xp + row) * ldw) + w);
            x.x += y.x;
            x.y += y.y;
        }
        if (nsplit > 1) *x0 = x;
        if (row < n_chol) {
            s.x += x.x * x.x - x.y * x.y;
            s.y += 2.0 * x.x * x.y;
        } else if (row == n_chol) {
            E1raw[w] = x;
        }
    }
    red[warp][lane] = s;
    __syncthreads();
    if (warp == 0) {
        double2 a = red[0][lane];
        for (int q = 1; q < 8; ++q) { a.x += red[q][lane].x; a.y += red[q][lane].y; }
        EJpart[(size_t)chunk * Wcap + w] = a;
    }
}

// ------------------------------------------------------------------------------------------------ S4: exchange
// Work item = (row tile of one pair, block of 64 walkers).  For the tile's rows K (singular vectors of pair (i,j)):
//   a[K][w] = sum_p U[K][p] Theta_j[p][w],  b[K][w] = sum_p W[K][p] Theta_i[p][w]   (two real FP64 GEMMs, DMMA)
//   e[w]   += wgt[K] * a[K][w] * b[K][w]  (complex product; wgt = -cK m_ij sigma_K)
// CTA tile <= 64 rows x 128 real columns x 2 accumulators, K tile 16.  Each of the 8 consumer warps owns ALL row
// fragments of the tile and 16 real columns (8 walkers), so any rank (nfrag = 1..8 fragments of 8 rows) is balanced
// over the warps and no cross-warp reduction is needed; the K loop is instantiated per nfrag (ex_kloop<NFRAG>) so a
// short tile issues no DMMA on padding (predicated-off DMMAs still occupy the pipe: seen with ncu on the paper-like
// small-rank workload).  4-stage TMA/mbarrier pipeline running across items; a tile of k fragments loads U and W as one
// box of 8 k rows each (a tensor map per box height).  The C fragment holds (re, im) of one walker in one lane, for a and b alike, so the complex
// product is lane-local; rows are reduced by warp shuffles.  Persistent CTAs with a static round-robin schedule and
// per-CTA partial sums accumulated in a fixed order -> bitwise repeatable.
constexpr int EX_STAGES = 4;
constexpr int EX_STAGE_BYTES = (2 * EX_BM + 2 * 128) * 128;
constexpr int EX_SMEM = EX_STAGES * EX_STAGE_BYTES + 1024 + 128 + EX_RING * 16;

// Which (tile, walker block) items a CTA works on, in which order.  Default: round robin over q = tile * NB + nb.  With a
// static schedule (small problems, where a CTA gets only a handful of items and one item more or less is a 5-15 % imbalance):
// tiles dealt to the CTAs by accumulated fragment count on the host (longest-processing-time first), CSR lists off / tile;
// every CTA runs its tiles in list order, all walker blocks of a tile one after the other.  Either way the order is fixed
// for a factor set and grid: results stay bitwise repeatable.
struct ExItems {
    const int* off;      // [gridDim.x + 1] or NULL (round robin)
    const int* tile;     // [n_tiles]
    __device__ __forceinline__ long long count(long long n_items, int NB) const {
        if (off) return (long long)(off[blockIdx.x + 1] - off[blockIdx.x]) * NB;
        return n_items > (long long)blockIdx.x ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    }
    __device__ __forceinline__ void at(long long it, int NB, int& tile_idx, int& nb) const {
        if (off) {
            tile_idx = tile[off[blockIdx.x] + (int)(it / NB)];
            nb = (int)(it % NB);
        } else {
            const long long q = blockIdx.x + it * gridDim.x;
            tile_idx = (int)(q / NB);
            nb = (int)(q % NB);
        }
    }
};

// COUL: also accumulate the two projections of the paper-literal compressed Coulomb term,
// aJ = U Theta_i and bJ = W Theta_j (Eq. 19/22 first term, "forming the projected vectors must occur four times",
// PAPER.md:181), from the same staged tiles; tiles are then cut at 4 fragments so the four accumulator sets fit.
template <int NFRAG, bool COUL, int MFMAX>
__device__ __forceinline__ void ex_kloop(int KT, uint32_t sbase, uint32_t full, uint32_t empty, int& cslot, uint32_t& cphase, int lane,
                                         const uint32_t (&xo)[4], uint32_t u_row, uint32_t tj_row, double (&accA)[MFMAX][2][2],
                                         double (&accB)[MFMAX][2][2], double (&accC)[COUL ? MFMAX : 1][2][2],
                                         double (&accD)[COUL ? MFMAX : 1][2][2]) {
    constexpr uint32_t W_OFF = EX_BM * 128, TI_OFF = 128 * 128;
    for (int kt = 0; kt < KT; ++kt) {
        if (kt) mbar_wait(full + 8 * cslot, cphase);     // the item's first stage was awaited by the caller
        const uint32_t st = sbase + cslot * EX_STAGE_BYTES;
#pragma unroll
        for (int ks = 0; ks < KTILE / 4; ++ks) {
            double a[NFRAG], w[NFRAG], bj[2], bi[2];
#pragma unroll
            for (int mf = 0; mf < NFRAG; ++mf) {
                a[mf] = lds_f64(st + u_row + mf * 1024 + xo[ks]);
                w[mf] = lds_f64(st + u_row + W_OFF + mf * 1024 + xo[ks]);
            }
#pragma unroll
            for (int nf = 0; nf < 2; ++nf) {
                bj[nf] = lds_f64(st + tj_row + nf * 1024 + xo[ks]);
                bi[nf] = lds_f64(st + tj_row + TI_OFF + nf * 1024 + xo[ks]);
            }
            if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
            for (int mf = 0; mf < NFRAG; ++mf)
#pragma unroll
                for (int nf = 0; nf < 2; ++nf) {
                    mma884(accA[mf][nf][0], accA[mf][nf][1], a[mf], bj[nf]);
                    mma884(accB[mf][nf][0], accB[mf][nf][1], w[mf], bi[nf]);
                    if constexpr (COUL) {
                        mma884(accC[mf][nf][0], accC[mf][nf][1], a[mf], bi[nf]);
                        mma884(accD[mf][nf][0], accD[mf][nf][1], w[mf], bj[nf]);
                    }
                }
        }
        if (++cslot == EX_STAGES) { cslot = 0; cphase ^= 1; }
    }
}

template <bool COUL, bool RAGGED>   // RAGGED: the batch is not a multiple of 64 walkers (warps without walkers skip their MMAs)
__global__ void __launch_bounds__(384, 1) k_exchange(const __grid_constant__ TmSet tmUs, const __grid_constant__ TmSet tmWs,
                                                     const __grid_constant__ CUtensorMap tmT, const double* __restrict__ wgt,
                                                     const ExTile* __restrict__ tiles, long long n_items, int NB, int N_pad, int ldw,
                                                     double* __restrict__ ekpart, double* __restrict__ ejpart, int Wcap, int n_w, ExItems items) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const uint32_t full = sbase + EX_STAGES * EX_STAGE_BYTES, empty = full + 8 * EX_STAGES;
    ExTile* ring = reinterpret_cast<ExTile*>(sgen + EX_STAGES * EX_STAGE_BYTES + 128);            // [EX_RING]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KT = N_pad / KTILE;
    double* mypart = ekpart + (size_t)blockIdx.x * 2 * Wcap;
    double* mypartJ = COUL ? ejpart + (size_t)blockIdx.x * 2 * Wcap : nullptr;
    for (int i = tid; i < 2 * Wcap; i += 384) {
        mypart[i] = 0.0;
        if constexpr (COUL) mypartJ[i] = 0.0;
    }
    if (tid == 0) {
        for (int k = 0; k < 8; ++k) { prefetch_tmap(&tmUs.m[k]); prefetch_tmap(&tmWs.m[k]); }
        prefetch_tmap(&tmT);
        for (int i = 0; i < EX_STAGES; ++i) { mbar_init(full + 8 * i, 1); mbar_init(empty + 8 * i, 8); }
        fence_barrier_init();
    }
    __syncthreads();
    if (warp < 4) {
        // ===== producer warpgroup; one lane drives TMA, running ahead of the consumers by up to EX_STAGES stages, across
        // work items.  The tile descriptor of item n is published in ring[n % EX_RING] before the item's first stage is armed.
        reg_dec_producer();
        if (warp == 0 && lane == 0) {
            int slot = 0, n = 0;
            uint32_t phase = 0;
            const long long my_items = items.count(n_items, NB);
            for (long long it = 0; it < my_items; ++it, ++n) {
                int tile_idx, nb;
                items.at(it, NB, tile_idx, nb);
                const ExTile tile = tiles[tile_idx];
                const uint32_t tx = (uint32_t)(2 * tile.nfrag * 8 + 2 * 128) * 128;
                for (int kt = 0; kt < KT; ++kt) {
                    mbar_wait(empty + 8 * slot, phase ^ 1);
                    if (kt == 0) ring[n % EX_RING] = tile;      // ordered before the consumers' wait by arrive.expect_tx (release)
                    const uint32_t st = sbase + slot * EX_STAGE_BYTES, bar = full + 8 * slot;
                    const int k0 = kt * KTILE;
                    mbar_expect_tx(bar, tx);
                    // one box of exactly the tile's rows per operand (tensor maps per box height 8 .. 64)
                    tma_load_2d(st, &tmUs.m[tile.nfrag - 1], k0, tile.row0, bar);
                    tma_load_2d(st + EX_BM * 128, &tmWs.m[tile.nfrag - 1], k0, tile.row0, bar);
                    tma_load_2d(st + 2 * EX_BM * 128, &tmT, k0, tile.pj * ldw + nb * 128, bar);
                    tma_load_2d(st + (2 * EX_BM + 128) * 128, &tmT, k0, tile.pi * ldw + nb * 128, bar);
                    if (++slot == EX_STAGES) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }
    // ===== 8 consumer warps (all row fragments x 16 real columns x 2 accumulators each)
    reg_inc_consumer();
    const int cw = warp - 4, g = lane >> 2, t = lane & 3;
    constexpr int MFMAX = COUL ? 4 : 8;
    double accA[MFMAX][2][2], accB[MFMAX][2][2], accC[COUL ? MFMAX : 1][2][2], accD[COUL ? MFMAX : 1][2][2];
#pragma unroll
    for (int a = 0; a < MFMAX; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            accA[a][b][0] = accA[a][b][1] = accB[a][b][0] = accB[a][b][1] = 0.0;
            if constexpr (COUL) accC[a][b][0] = accC[a][b][1] = accD[a][b][0] = accD[a][b][1] = 0.0;
        }
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t u_row = (uint32_t)g * 128;
    const uint32_t tj_row = (uint32_t)(2 * EX_BM + cw * 16 + g) * 128;
    int cslot = 0, n = 0;
    uint32_t cphase = 0;
    const long long my_items = items.count(n_items, NB);
    for (long long it = 0; it < my_items; ++it, ++n) {
        int tile_idx, nb;
        items.at(it, NB, tile_idx, nb);
        // this lane's slice of the CTA partial (lanes with g == 0 own walker cw*8 + nf*4 + t of the block): fetched now,
        // updated after the K loop (same thread wrote it last, so program order makes the previous update visible)
        double2* myp = reinterpret_cast<double2*>(mypart + (size_t)nb * 128 + cw * 16 + 2 * t);
        double2* mypJ = reinterpret_cast<double2*>(mypartJ + (size_t)nb * 128 + cw * 16 + 2 * t);
        double2 prev[2], prevJ[2];
        if (g == 0) {
            prev[0] = myp[0]; prev[1] = myp[4];
            if constexpr (COUL) { prevJ[0] = mypJ[0]; prevJ[1] = mypJ[4]; }
        }
        mbar_wait(full + 8 * cslot, cphase);            // first stage of the item: its descriptor is in the ring now
        const ExTile tile = ring[n % EX_RING];
        if (RAGGED && nb * WALKER_TILE + cw * 8 >= n_w) {
            // none of this warp's 8 walkers exists (ragged last block, batches below 64 walkers): no MMAs, only hand the
            // stages back; the warps that do have walkers then get the tensor pipe of their scheduler to themselves
            for (int kt = 0; kt < KT; ++kt) {
                if (kt) mbar_wait(full + 8 * cslot, cphase);
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + 8 * cslot);
                if (++cslot == EX_STAGES) { cslot = 0; cphase ^= 1; }
            }
            continue;
        }
#define LO_EX_CASE(NF_) ex_kloop<NF_, COUL, MFMAX>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, tj_row, accA, accB, accC, accD)
        if constexpr (COUL) {
            switch (tile.nfrag) {                       // warp- and CTA-uniform; COUL tiles have at most 4 fragments
                case 1: LO_EX_CASE(1); break;
                case 2: LO_EX_CASE(2); break;
                case 3: LO_EX_CASE(3); break;
                default: LO_EX_CASE(4); break;
            }
        } else {
            switch (tile.nfrag) {
                case 1: LO_EX_CASE(1); break;
                case 2: LO_EX_CASE(2); break;
                case 3: LO_EX_CASE(3); break;
                case 4: LO_EX_CASE(4); break;
                case 5: LO_EX_CASE(COUL ? 4 : 5); break;
                case 6: LO_EX_CASE(COUL ? 4 : 6); break;
                case 7: LO_EX_CASE(COUL ? 4 : 7); break;
                default: LO_EX_CASE(COUL ? 4 : 8); break;
            }
        }
#undef LO_EX_CASE
        // fused epilogue: e[w] = sum over this lane's rows of weight * a * b (complex), then over the 8 row groups of
        // the warp (shuffles), in a fixed order; fragments beyond nfrag hold zeros
        double e[2][2], eJ[2][2];
#pragma unroll
        for (int nf = 0; nf < 2; ++nf) e[nf][0] = e[nf][1] = eJ[nf][0] = eJ[nf][1] = 0.0;
#pragma unroll
        for (int mf = 0; mf < MFMAX; ++mf) {
            const double wv = (mf < tile.nfrag) ? __ldg(wgt + tile.row0 + mf * 8 + g) : 0.0;
#pragma unroll
            for (int nf = 0; nf < 2; ++nf) {
                double ar = accA[mf][nf][0], ai = accA[mf][nf][1], br = accB[mf][nf][0], bi = accB[mf][nf][1];
                e[nf][0] = fma(wv, ar * br - ai * bi, e[nf][0]);
                e[nf][1] = fma(wv, ar * bi + ai * br, e[nf][1]);
                accA[mf][nf][0] = accA[mf][nf][1] = accB[mf][nf][0] = accB[mf][nf][1] = 0.0;
                if constexpr (COUL) {
                    ar = accC[mf][nf][0]; ai = accC[mf][nf][1]; br = accD[mf][nf][0]; bi = accD[mf][nf][1];
                    eJ[nf][0] = fma(wv, ar * br - ai * bi, eJ[nf][0]);
                    eJ[nf][1] = fma(wv, ar * bi + ai * br, eJ[nf][1]);
                    accC[mf][nf][0] = accC[mf][nf][1] = accD[mf][nf][0] = accD[mf][nf][1] = 0.0;
                }
            }
        }
#pragma unroll
        for (int nf = 0; nf < 2; ++nf)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                double v = e[nf][c];
                v += __shfl_xor_sync(0xffffffffu, v, 4);
                v += __shfl_xor_sync(0xffffffffu, v, 8);
                v += __shfl_xor_sync(0xffffffffu, v, 16);
                e[nf][c] = v;
                if constexpr (COUL) {
                    v = eJ[nf][c];
                    v += __shfl_xor_sync(0xffffffffu, v, 4);
                    v += __shfl_xor_sync(0xffffffffu, v, 8);
                    v += __shfl_xor_sync(0xffffffffu, v, 16);
                    eJ[nf][c] = v;
                }
            }
        if (g == 0) {
            myp[0] = make_double2(prev[0].x + e[0][0], prev[0].y + e[0][1]);
            myp[4] = make_double2(prev[1].x + e[1][0], prev[1].y + e[1][1]);
            if constexpr (COUL) {
                mypJ[0] = make_double2(prevJ[0].x + eJ[0][0], prevJ[0].y + eJ[0][1]);
                mypJ[4] = make_double2(prevJ[1].x + eJ[1][0], prevJ[1].y + eJ[1][1]);
            }
        }
    }
}

// ---- narrow-batch exchange (n_w <= 32, e.g. the paper's 16 walkers per GPU): a 64-walker column block
// would leave 6 of the 8 consumer warps without walkers, so here a work item is (row tile, block of 16 walkers = 32 real
// columns = 4 column tiles of the m8n8k4 MMA) and the work units are (row fragment, column tile): consumer warp cw owns
// column tile cw & 3 (4 walkers) and the fragments (cw >> 2), (cw >> 2) + 2, ... of the tile.  The two warps of a
// scheduler (cw, cw + 4) then hold nfrag units between them whatever nfrag is, so the four tensor pipes carry equal
// loads (the first version split fragments cw >> 1 and 4 + (cw >> 1): 3 units on two schedulers, 2 on the others at
// nfrag = 5).  The K loop is instantiated per fragment count of the warp (no padding MMAs).  The weighted complex dots
// are accumulated IN REGISTERS across all items of the CTA (an item only adds lane-local terms: no shuffle, no barrier,
// no shared memory per item); one shuffle reduction over the row groups and one fixed-order addition of the two
// fragment groups at the end of the kernel.  Same TMA/mbarrier pipeline; U and W arrive as ONE box of exactly the
// tile's rows each (tensor maps per box height).
constexpr int EN_STAGES = 6;
constexpr int EN_STAGE_BYTES = (2 * EX_BM + 2 * 32) * 128;
constexpr int EN_SMEM = EN_STAGES * EN_STAGE_BYTES + 1024 + 128 + EX_RING * 16 + 2 * 64 * 8;

template <int NFW>   // fragments of this warp in the current tile (0..4)
__device__ __forceinline__ void en_kloop(int KT, uint32_t sbase, uint32_t full, uint32_t empty, int& cslot, uint32_t& cphase, int lane,
                                         const uint32_t (&xo)[4], uint32_t u_row, uint32_t tj_row, double (&accA)[4][2], double (&accB)[4][2]) {
    constexpr uint32_t W_OFF = EX_BM * 128, TI_OFF = 32 * 128;
    for (int kt = 0; kt < KT; ++kt) {
        if (kt) mbar_wait(full + 8 * cslot, cphase);     // the item's first stage was awaited by the caller
        if constexpr (NFW == 0) {
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + 8 * cslot);
        } else {
            const uint32_t st = sbase + cslot * EN_STAGE_BYTES;
#pragma unroll
            for (int ks = 0; ks < KTILE / 4; ++ks) {
                double a[NFW], w[NFW];
#pragma unroll
                for (int j = 0; j < NFW; ++j) {
                    a[j] = lds_f64(st + u_row + j * 2048 + xo[ks]);            // fragments two apart: 16 rows = 2048 bytes
                    w[j] = lds_f64(st + u_row + W_OFF + j * 2048 + xo[ks]);
                }
                const double bj = lds_f64(st + tj_row + xo[ks]), bi = lds_f64(st + tj_row + TI_OFF + xo[ks]);
                if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                for (int j = 0; j < NFW; ++j) {
                    mma884(accA[j][0], accA[j][1], a[j], bj);
                    mma884(accB[j][0], accB[j][1], w[j], bi);
                }
            }
        }
        if (++cslot == EN_STAGES) { cslot = 0; cphase ^= 1; }
    }
}

__global__ void __launch_bounds__(384, 1) k_exchange_narrow(const __grid_constant__ TmSet tmUs, const __grid_constant__ TmSet tmWs,
                                                            const __grid_constant__ CUtensorMap tmT32, const double* __restrict__ wgt,
                                                            const ExTile* __restrict__ tiles, long long n_items, int NB, int N_pad, int ldw,
                                                            double* __restrict__ ekpart, int Wcap, ExItems items) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const uint32_t full = sbase + EN_STAGES * EN_STAGE_BYTES, empty = full + 8 * EN_STAGES;
    ExTile* ring = reinterpret_cast<ExTile*>(sgen + EN_STAGES * EN_STAGE_BYTES + 128);
    double* red = reinterpret_cast<double*>(sgen + EN_STAGES * EN_STAGE_BYTES + 128 + EX_RING * 16);      // [2 fragment groups][2 blocks x 32 columns]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KT = N_pad / KTILE;
    double* mypart = ekpart + (size_t)blockIdx.x * 2 * Wcap;
    for (int i = tid; i < 2 * Wcap; i += 384) mypart[i] = 0.0;
    if (tid == 0) {
        for (int k = 0; k < 8; ++k) { prefetch_tmap(&tmUs.m[k]); prefetch_tmap(&tmWs.m[k]); }
        prefetch_tmap(&tmT32);
        for (int i = 0; i < EN_STAGES; ++i) { mbar_init(full + 8 * i, 1); mbar_init(empty + 8 * i, 8); }
        fence_barrier_init();
    }
    __syncthreads();
    if (warp < 4) {
        reg_dec_producer();
        if (warp == 0 && lane == 0) {
            int slot = 0, n = 0;
            uint32_t phase = 0;
            const long long my_items = items.count(n_items, NB);
            for (long long it = 0; it < my_items; ++it, ++n) {
                int tile_idx, nb;
                items.at(it, NB, tile_idx, nb);
                const ExTile tile = tiles[tile_idx];
                const uint32_t tx = (uint32_t)(2 * tile.nfrag * 8 + 2 * 32) * 128;
                const CUtensorMap* mu = &tmUs.m[tile.nfrag - 1];
                const CUtensorMap* mw = &tmWs.m[tile.nfrag - 1];
                for (int kt = 0; kt < KT; ++kt) {
                    mbar_wait(empty + 8 * slot, phase ^ 1);
                    if (kt == 0) ring[n % EX_RING] = tile;
                    const uint32_t st = sbase + slot * EN_STAGE_BYTES, bar = full + 8 * slot;
                    const int k0 = kt * KTILE;
                    mbar_expect_tx(bar, tx);
                    tma_load_2d(st, mu, k0, tile.row0, bar);
                    tma_load_2d(st + EX_BM * 128, mw, k0, tile.row0, bar);
                    tma_load_2d(st + 2 * EX_BM * 128, &tmT32, k0, tile.pj * ldw + nb * 32, bar);
                    tma_load_2d(st + 2 * EX_BM * 128 + 32 * 128, &tmT32, k0, tile.pi * ldw + nb * 32, bar);
                    if (++slot == EN_STAGES) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }
    reg_inc_consumer();
    const int cw = warp - 4, g = lane >> 2, t = lane & 3, ctid = tid - 128;
    const int nt = cw & 3, fg = cw >> 2;           // column tile (walkers 4 nt .. 4 nt + 3 of the block), fragment group
    double accA[4][2], accB[4][2];
#pragma unroll
    for (int j = 0; j < 4; ++j) accA[j][0] = accA[j][1] = accB[j][0] = accB[j][1] = 0.0;
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t u_row = (uint32_t)(fg * 8 + g) * 128;
    const uint32_t tj_row = (uint32_t)(2 * EX_BM + nt * 8 + g) * 128;
    double e0r = 0.0, e0i = 0.0, e1r = 0.0, e1i = 0.0;      // this lane's running sums for walker block 0 / 1
    int cslot = 0, n = 0;
    uint32_t cphase = 0;
    const long long my_items = items.count(n_items, NB);
    for (long long it = 0; it < my_items; ++it, ++n) {
        int tile_idx, nb;
        items.at(it, NB, tile_idx, nb);
        mbar_wait(full + 8 * cslot, cphase);
        const ExTile tile = ring[n % EX_RING];
        const int nfw = tile.nfrag > fg ? (tile.nfrag - fg + 1) >> 1 : 0;     // warp-uniform
        switch (nfw) {
            case 0: en_kloop<0>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, tj_row, accA, accB); break;
            case 1: en_kloop<1>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, tj_row, accA, accB); break;
            case 2: en_kloop<2>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, tj_row, accA, accB); break;
            case 3: en_kloop<3>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, tj_row, accA, accB); break;
            default: en_kloop<4>(KT, sbase, full, empty, cslot, cphase, lane, xo, u_row, tj_row, accA, accB); break;
        }
        double er = 0.0, ei = 0.0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const double wv = j < nfw ? __ldg(wgt + tile.row0 + (fg + 2 * j) * 8 + g) : 0.0;
            const double ar = accA[j][0], ai = accA[j][1], br = accB[j][0], bi = accB[j][1];
            er = fma(wv, ar * br - ai * bi, er);
            ei = fma(wv, ar * bi + ai * br, ei);
            accA[j][0] = accA[j][1] = accB[j][0] = accB[j][1] = 0.0;
        }
        if (nb == 0) { e0r += er; e0i += ei; }
        else { e1r += er; e1i += ei; }
    }
    // ---- once per kernel: rows (shuffles over g), then the two fragment groups in a fixed order
    double v[4] = {e0r, e0i, e1r, e1i};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        v[c] += __shfl_xor_sync(0xffffffffu, v[c], 4);
        v[c] += __shfl_xor_sync(0xffffffffu, v[c], 8);
        v[c] += __shfl_xor_sync(0xffffffffu, v[c], 16);
    }
    if (g == 0) {
        double* r = red + fg * 64 + nt * 8 + 2 * t;
        r[0] = v[0]; r[1] = v[1]; r[32] = v[2]; r[33] = v[3];
    }
    bar_sync_consumers();
    if (ctid < 32 * NB) mypart[ctid] = red[ctid] + red[64 + ctid];
}

// ------------------------------------------------------------------------------------------------ NEXT-1: propagator
// x[w][g] (complex128, walker-major) -> XT[2w + c][g] (K-major real operand of the propagator GEMM); the K padding
// columns g >= n_chol stay zero from allocation.  grid (ceil(n_chol/128), n_w), block 128.
__global__ void __launch_bounds__(128) k_pack_x(const double2* __restrict__ x, double* __restrict__ XT, int n_chol, int Xk_pad) {
    const int g = blockIdx.x * 128 + threadIdx.x, w = blockIdx.y;
    if (g >= n_chol) return;
    const double2 v = x[(size_t)w * n_chol + g];
    XT[(size_t)(2 * w) * Xk_pad + g] = v.x;
    XT[(size_t)(2 * w + 1) * Xk_pad + g] = v.y;
}

// ------------------------------------------------------------------------------------------------ S5: combine
__global__ void k_finalize(const double2* __restrict__ EJpart, int n_chunks, const double2* __restrict__ E1raw,
                           const double2* __restrict__ EKpart, int n_ctas, const int* __restrict__ status, int n_spin, int Wcap,
                           int n_w, double c1, double cJ, double2* __restrict__ E_L, double2* __restrict__ E1, double2* __restrict__ E_J,
                           double2* __restrict__ E_K, int* __restrict__ st_out, double2* __restrict__ Eout4,
                           const double2* __restrict__ EJLpart) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_w) return;
    double2 ej = make_double2(0.0, 0.0), ek = make_double2(0.0, 0.0);
    for (int c = 0; c < n_chunks; ++c) { double2 v = EJpart[(size_t)c * Wcap + w]; ej.x += v.x; ej.y += v.y; }
    for (int b = 0; b < n_ctas; ++b) { double2 v = EKpart[(size_t)b * Wcap + w]; ek.x += v.x; ek.y += v.y; }
    double2 e1 = E1raw[w];
    e1.x *= c1; e1.y *= c1;
    ej.x *= cJ; ej.y *= cJ;
    if (EJLpart) {
        // paper-literal compressed Coulomb term (Eq. 19/22): E_J^LO = 2 sum_{i<=j} m_ij sum_K sigma_K aJ_K bJ_K = -2 sum(wgt aJ bJ)
        ej = make_double2(0.0, 0.0);
        for (int b = 0; b < n_ctas; ++b) { double2 v = EJLpart[(size_t)b * Wcap + w]; ej.x += v.x; ej.y += v.y; }
        ej.x *= -2.0; ej.y *= -2.0;
    }
    int bad = status[w];
    if (n_spin == 2) bad |= status[Wcap + w];
    if (bad) {
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        e1 = ej = ek = make_double2(nan, nan);
    }
    double2 el = make_double2(e1.x + ej.x + ek.x, e1.y + ej.y + ek.y);
    if (E_L) E_L[w] = el;
    if (E1) E1[w] = e1;
    if (E_J) E_J[w] = ej;
    if (E_K) E_K[w] = ek;
    if (st_out) st_out[w] = bad;
    if (Eout4) { Eout4[4 * w] = el; Eout4[4 * w + 1] = e1; Eout4[4 * w + 2] = ej; Eout4[4 * w + 3] = ek; }
}

int pick_split(long long base_items, int ksteps, int sms) {
    int best = 1;
    double best_eff = -1;
    for (int s = 1; s <= MAX_SPLIT; ++s) {
        if (ksteps / s < 8 && s > 1) break;
        long long items = base_items * s;
        long long waves = (items + sms - 1) / sms;
        double eff = (double)items / (double)(waves * sms);
        if (eff > best_eff + 0.02) { best_eff = eff; best = s; }
    }
    return best;
}

typedef void (*OvFn)(const double*, const double2*, double2*, int, int, int);
template <int M>
OvFn ov_fn_n(int nfw) {
    switch (nfw) {
        case 1: return k_overlap<M, 1>;
        case 2: return k_overlap<M, 2>;
        case 3: return k_overlap<M, 3>;
        case 4: return k_overlap<M, 4>;
        case 5: return k_overlap<M, 5>;
        case 6: return k_overlap<M, 6>;
        case 7: return k_overlap<M, 7>;
        default: return k_overlap<M, 8>;
    }
}
OvFn ov_fn(int mfb, int nfw) {
    switch (mfb) {
        case 1: return ov_fn_n<1>(nfw);
        case 2: return ov_fn_n<2>(nfw);
        case 3: return ov_fn_n<3>(nfw);
        case 4: return ov_fn_n<4>(nfw);
        default: return ov_fn_n<5>(nfw);
    }
}
typedef void (*ThFn)(const double2*, const double2*, double*, int, int, int, int, int);
template <int M>
ThFn th_fn_t() { return k_theta<M>; }
ThFn th_fn(int mfb) {
    static const ThFn tab[16] = {th_fn_t<1>(), th_fn_t<2>(), th_fn_t<3>(), th_fn_t<4>(), th_fn_t<5>(), th_fn_t<6>(), th_fn_t<7>(), th_fn_t<8>(),
                                 th_fn_t<9>(), th_fn_t<10>(), th_fn_t<11>(), th_fn_t<12>(), th_fn_t<13>(), th_fn_t<14>(), th_fn_t<15>(), th_fn_t<16>()};
    return tab[mfb - 1];
}

}  // namespace

lo_status configure_kernels() {
    cudaError_t e;
    e = cudaFuncSetAttribute(k_coulomb<false, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, CO_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_coulomb<true, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, CO_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_coulomb<true, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, CO_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_coulomb<true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, CO_SMEM);
    if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_coulomb): ") + cudaGetErrorString(e)); return LO_ECUDA; }
    e = cudaFuncSetAttribute(k_exchange<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, EX_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_exchange<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, EX_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_exchange<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, EX_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_exchange<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, EX_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_exchange_narrow, cudaFuncAttributeMaxDynamicSharedMemorySize, EN_SMEM);
    if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_exchange): ") + cudaGetErrorString(e)); return LO_ECUDA; }
    e = cudaFuncSetAttribute(k_inverse<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_inverse): ") + cudaGetErrorString(e)); return LO_ECUDA; }
    for (int m = 1; m <= 16; ++m) {
        e = cudaFuncSetAttribute((const void*)th_fn(m), cudaFuncAttributeMaxDynamicSharedMemorySize, 120 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)th_fn(m), cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_theta): ") + cudaGetErrorString(e)); return LO_ECUDA; }
    }
    for (int m = 1; m <= 5; ++m)
        for (int n = 1; n <= 8; ++n) {
            e = cudaFuncSetAttribute((const void*)ov_fn(m, n), cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
            if (e == cudaSuccess) e = cudaFuncSetAttribute((const void*)ov_fn(m, n), cudaFuncAttributePreferredSharedMemoryCarveout, 100);
            if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_overlap): ") + cudaGetErrorString(e)); return LO_ECUDA; }
        }
    if (configure_cas_kernels() != LO_OK) return LO_ECUDA;
    e = cudaFuncSetAttribute(k_inverse<true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_inverse): ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

// S1 of one spin block: A = Psi^T Phi (Psi = the first O columns of a [N][ldpsi] orbital matrix), A^-1 with per-walker
// status, Theta^T panels written to `thT` (panel stride ldw_t) starting at panel o_base.
void launch_s1(lo_factors* f, int n_w, const double* psi, int ldpsi, int O, const void* phi, double* dA, int* status, double* thT,
               int o_base, int ldw_t, cudaStream_t stream) {
    const int N = f->N, N_pad = f->N_pad;
    {
        Timer tm(f, stream, LO_K_OVERLAP);
        const int NF = (2 * O + 7) / 8, nfw = (std::min(NF, OV_NFB) + 7) / 8;
        const int MF = (O + 7) / 8, n_mb = (MF + 4) / 5, mfb = (MF + n_mb - 1) / n_mb;     // row blocks of <= 5 fragments
        dim3 grid(n_mb, n_w, (NF + OV_NFB - 1) / OV_NFB);
        const size_t smem = (size_t)2 * OV_PC * (OV_LDA + ov_ldb(O)) * 8;      // two staging buffers
        ov_fn(mfb, nfw)<<<grid, 256, smem, stream>>>(psi, (const double2*)phi, (double2*)dA, N, O, ldpsi);
    }
    {
        Timer tm(f, stream, LO_K_INVERSE);
        size_t aux = (size_t)(2 * O + 1) * 16 + (size_t)((O + 3) & ~3) * 4 + 16;
        size_t need = aux + (size_t)O * O * 16;
        const int rt = (O + 15) / 16;
        double2* Ad = (double2*)dA;
        // register-resident variant while >= 2 CTAs per SM fit (<= 96 registers: O <= 48); beyond that its serial chain
        // (pivot search, reciprocal, 3 barriers) is no longer hidden by a second CTA and the shared-memory kernel wins
        if (rt == 1) k_inverse_reg<1><<<n_w, 256, 0, stream>>>(Ad, status, O);
        else if (rt == 2) k_inverse_reg<2><<<n_w, 256, 0, stream>>>(Ad, status, O);
        else if (rt == 3) k_inverse_reg<3><<<n_w, 256, 0, stream>>>(Ad, status, O);
        else if (need <= 200 * 1024)
            k_inverse<true><<<n_w, 256, need, stream>>>(Ad, status, O);
        else
            k_inverse<false><<<n_w, 256, aux, stream>>>(Ad, status, O);
    }
    {
        Timer tm(f, stream, LO_K_THETA);
        const int MF = (2 * O + 7) / 8, n_mb = (MF + 15) / 16, mfb = (MF + n_mb - 1) / n_mb;
        dim3 grid((N_pad + 63) / 64, n_mb, n_w);
        th_fn(mfb)<<<grid, 256, (size_t)2 * (mfb * 8 + 64) * TH_LD * 8, stream>>>((const double2*)phi, (const double2*)dA, thT, N, N_pad, O, o_base, ldw_t);
    }
}

lo_status launch_local_energy(lo_factors* f, int n_w, const void* phi_a, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K,
                              int* walker_status, void* Eout4, cudaStream_t stream) {
    const void* phis[2] = {phi_a, phi_b};
    for (int s = 0; s < f->n_spin; ++s)
        launch_s1(f, n_w, f->ops->dPsi[s], f->n_occ[s], f->n_occ[s], phis[s], f->dA[s], f->dStatus + (size_t)s * f->Wcap, f->dThT, f->o_base[s],
                  f->ldw, stream);
    return launch_s3_s5(f, n_w, E_L, E1, E_J, E_K, walker_status, Eout4, stream);
}

// S2 + S3 on the Theta^T panels of n_w walkers: X^g_w (and the hbar row) into f->dXpart, then k_ej.
void launch_coulomb_x(lo_factors* f, int n_w, cudaStream_t stream) {
    const int N_pad = f->N_pad, ldw = f->ldw, Wcap = f->Wcap;
    const int NB = (n_w + WALKER_TILE - 1) / WALKER_TILE;
    const int RB = f->Xp / CO_BM;
    const int ksteps = f->O_tot * (N_pad / KTILE);
    const int nsplit = pick_split((long long)RB * NB, ksteps, f->num_sms);
    double2* EJpart = (double2*)f->dEJpart;
    double2* E1raw = EJpart + (size_t)RB * Wcap;
    {
        Timer tm(f, stream, LO_K_COULOMB);
        long long items = (long long)RB * NB * nsplit;
        int grid = (int)std::min<long long>(items, f->num_sms);
        if (n_w <= 16)
            k_coulomb<true, 1><<<grid, 384, CO_SMEM, stream>>>(f->ops->tmLbar, f->tmTheta, f->tmTheta32, f->dXpart, f->Xp, f->O_tot, N_pad, ldw, RB, NB, nsplit, 2 * n_w);
        else if (n_w <= 32)
            k_coulomb<true, 2><<<grid, 384, CO_SMEM, stream>>>(f->ops->tmLbar, f->tmTheta, f->tmTheta32, f->dXpart, f->Xp, f->O_tot, N_pad, ldw, RB, NB, nsplit, 2 * n_w);
        else if (n_w % WALKER_TILE)
            k_coulomb<true, 4><<<grid, 384, CO_SMEM, stream>>>(f->ops->tmLbar, f->tmTheta, f->tmTheta32, f->dXpart, f->Xp, f->O_tot, N_pad, ldw, RB, NB, nsplit, 2 * n_w);
        else
            k_coulomb<false, 4><<<grid, 384, CO_SMEM, stream>>>(f->ops->tmLbar, f->tmTheta, f->tmTheta32, f->dXpart, f->Xp, f->O_tot, N_pad, ldw, RB, NB, nsplit, 2 * n_w);
        dim3 g2(NB * 2, RB);
        k_ej<<<g2, 256, 0, stream>>>(f->dXpart, EJpart, E1raw, f->Xp, ldw, nsplit, f->n_chol, Wcap);
    }
}

void launch_gemm_kmajor(const CUtensorMap& tmA, const CUtensorMap& tmB, double* out, long long rows, long long cols, int N_pad, long long ld_out,
                        int num_sms, cudaStream_t stream) {
    const int RB = (int)(rows / CO_BM), NB = (int)(cols / 128);
    const long long items = (long long)RB * NB;
    const int grid = (int)std::min<long long>(std::max<long long>(items, 1), num_sms);
    k_coulomb<false, 4><<<grid, 384, CO_SMEM, stream>>>(tmA, tmB, tmB, out, (int)rows, 1, N_pad, (int)ld_out, RB, NB, 1, (int)cols);
}

// S2-S5 on the Theta^T panels of n_w (possibly virtual, see lo_local_energy_cas) walkers.
lo_status launch_s3_s5(lo_factors* f, int n_w, void* E_L, void* E1, void* E_J, void* E_K, int* walker_status, void* Eout4, cudaStream_t stream) {
    const int N_pad = f->N_pad, ldw = f->ldw, Wcap = f->Wcap;
    const int NB = (n_w + WALKER_TILE - 1) / WALKER_TILE;
    // ---- S2 + S3
    const bool i8 = f->ex_mode == LO_EXCHANGE_INT8;
    if (i8) {
        // INT8 route (lo_exchange_i8.cu): digits of Theta^T once per call, X^g_w from exact INT8 digit products on tcgen05, then k_ej
        Timer tm(f, stream, LO_K_COULOMB);
        launch_slice_theta_i8(f, n_w, stream);
        const int nsplit = launch_coulomb_i8(f, n_w, stream);
        dim3 g2(NB * 2, f->Xp / CO_BM);
        k_ej<<<g2, 256, 0, stream>>>(f->dXpart, (double2*)f->dEJpart, (double2*)f->dEJpart + (size_t)(f->Xp / CO_BM) * Wcap, f->Xp, ldw, nsplit, f->n_chol, Wcap);
    } else
        launch_coulomb_x(f, n_w, stream);
    const int RB = f->Xp / CO_BM;
    double2* EJpart = (double2*)f->dEJpart;
    double2* E1raw = EJpart + (size_t)RB * Wcap;
    // ---- S4
    int ex_grid = 0;
    const double* ek_part = f->dEKpart;
    const double* ejl_part = f->coulomb_lo ? f->dEJLpart : nullptr;
    {
        Timer tm(f, stream, LO_K_EXCHANGE);
        const bool coul = f->coulomb_lo != 0;
        long long items = (coul ? f->n_tiles4 : f->n_tiles) * NB;
        ex_grid = (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
        const bool ragged = n_w % WALKER_TILE != 0;
        // small problems: static LPT schedule of the tiles (grid = all SMs); large ones: round robin in L2-block order
        const ExItems rr = {nullptr, nullptr}, lpt = {f->dSchedOff, f->dSchedTile};
        if (i8) {
            // fp64-accurate projections from INT8 digit slices on the tcgen05 tensor cores (lo_exchange_i8.cu)
            launch_exchange_i8(f, n_w, stream, coul, &ek_part, &ex_grid, &ejl_part);
        } else if (!coul && n_w <= 32) {
            // narrow batch: 16-walker column blocks, row fragments split over the warps
            const int NB16 = (n_w + 15) / 16;
            items = f->n_tiles * NB16;
            const bool use_lpt = items <= 64LL * f->num_sms && f->n_tiles >= 8LL * f->num_sms;     // whole tiles are dealt: needs many tiles per CTA
            ex_grid = use_lpt ? f->num_sms : (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
            k_exchange_narrow<<<ex_grid, 384, EN_SMEM, stream>>>(f->tmUf, f->tmWf, f->tmTheta32, f->dWgt, f->dTiles, items, NB16,
                                                                 N_pad, ldw, f->dEKpart, Wcap, use_lpt ? lpt : rr);
        } else
#define LO_EX_LAUNCH(C_, R_, TILES_, EJ_)                                                                                              \
    k_exchange<C_, R_><<<ex_grid, 384, EX_SMEM, stream>>>(f->tmUf, f->tmWf, f->tmTheta, f->dWgt, TILES_, items, NB, N_pad, ldw, \
                                                          f->dEKpart, EJ_, Wcap, n_w, IT_)
        {
            const bool use_lpt = !coul && items <= 64LL * f->num_sms && f->n_tiles >= 8LL * f->num_sms;
            if (use_lpt) ex_grid = f->num_sms;
            const ExItems IT_ = use_lpt ? lpt : rr;
            if (coul && ragged) LO_EX_LAUNCH(true, true, f->dTiles4, f->dEJLpart);
            else if (coul) LO_EX_LAUNCH(true, false, f->dTiles4, f->dEJLpart);
            else if (ragged) LO_EX_LAUNCH(false, true, f->dTiles, nullptr);
            else LO_EX_LAUNCH(false, false, f->dTiles, nullptr);
        }
#undef LO_EX_LAUNCH
    }
    // ---- S5
    {
        Timer tm(f, stream, LO_K_FINAL);
        const double c1 = f->n_spin == 1 ? 2.0 : 1.0, cJ = f->n_spin == 1 ? 2.0 : 0.5;
        k_finalize<<<(n_w + 127) / 128, 128, 0, stream>>>(EJpart, RB, E1raw, (const double2*)ek_part, ex_grid, f->dStatus, f->n_spin, Wcap,
                                                          n_w, c1, cJ, (double2*)E_L, (double2*)E1, (double2*)E_J, (double2*)E_K,
                                                          walker_status, (double2*)Eout4,
                                                          (const double2*)ejl_part);
    }
    f->last_n_w = n_w;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("kernel launch failed: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

// B[r(p,q)][w] = sum_g L^g_pq x^g_w: the Coulomb GEMM kernel with A = Lt (K = g), one "orbital panel",
// no split-K (N(N+1)/2 / 128 row blocks fill the machine), output straight into dB.
lo_status launch_propagator(lo_factors* f, int n_w, const void* x_dev, cudaStream_t stream) {
    SharedOps& ops = *f->ops;
    const int NB = (n_w + WALKER_TILE - 1) / WALKER_TILE;
    const int RB = (int)(ops.tri_pad / CO_BM);
    {
        Timer tm(f, stream, LO_K_PROPAGATOR);
        dim3 g1((f->n_chol + 127) / 128, n_w);
        k_pack_x<<<g1, 128, 0, stream>>>((const double2*)x_dev, f->dXT, f->n_chol, ops.Xk_pad);
        const long long items = (long long)RB * NB;
        const int grid = (int)std::min<long long>(items, f->num_sms);
        if (f->ex_mode == LO_EXCHANGE_INT8 && f->dLtq)
            launch_propagator_i8(f, n_w, stream);          // exact INT8 digit products on tcgen05 (lo_exchange_i8.cu)
        else if (n_w % WALKER_TILE)
            k_coulomb<true, 4><<<grid, 384, CO_SMEM, stream>>>(ops.tmLt, f->tmXT, f->tmXT, f->dB, (int)ops.tri_pad, 1, ops.Xk_pad, f->ldw, RB, NB, 1, 2 * n_w);
        else
            k_coulomb<false, 4><<<grid, 384, CO_SMEM, stream>>>(ops.tmLt, f->tmXT, f->tmXT, f->dB, (int)ops.tri_pad, 1, ops.Xk_pad, f->ldw, RB, NB, 1, 2 * n_w);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("lo_propagator: kernel launch failed: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

}  // namespace lo

// ------------------------------------------------------------------------------------------------ allocation-free S1
// lo_theta_noalloc (include/lo_afqmc.h): step S1 for callers that cannot allocate.  The scratch of the S1 kernels -- the
// overlap matrices, inverted in place -- is this file-scope array; every GPU that loads the library holds it until exit.
// In host code the NAME below is a host-side stand-in, not a device address: the kernels get the pointer that
// cudaGetSymbolAddress returned for the device they run on (fetched once per device, with that device current).
static __device__ __align__(256) unsigned char lo_noalloc_scratch[LO_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
double* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {nullptr};     // device address of lo_noalloc_scratch, per device
}  // namespace

extern "C" lo_status lo_theta_noalloc_init(int device) {
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev || device >= NOALLOC_MAX_DEVICES) {
        (void)cudaGetLastError();
        lo::set_error("lo_theta_noalloc_init: no such CUDA device");
        return LO_EINVAL;
    }
    if (g_noalloc_ptr[device]) return LO_OK;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) { lo::set_error(std::string("lo_theta_noalloc_init: cudaSetDevice: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    if (lo::configure_kernels() != LO_OK) return LO_ECUDA;      // shared-memory attributes of the S1 kernels (no allocation)
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, lo_noalloc_scratch);
    if (e != cudaSuccess || !p) {
        lo::set_error(std::string("lo_theta_noalloc_init: cudaGetSymbolAddress(lo_noalloc_scratch): ") + cudaGetErrorString(e));
        return LO_ECUDA;
    }
    g_noalloc_ptr[device] = static_cast<double*>(p);
    return LO_OK;
}

extern "C" lo_status lo_theta_noalloc(int device, int N, int n_occ, int n_w, const double* psi_dev, const void* phi_dev, double* thetaT_dev,
                                      int ld_w, int* status_dev, void* stream) {
    if (N <= 0 || n_occ <= 0 || n_occ > N || n_w <= 0 || !psi_dev || !phi_dev || !thetaT_dev || !status_dev || ld_w < 2 * n_w || (ld_w & 1)) {
        lo::set_error("lo_theta_noalloc: invalid argument (need 1 <= n_occ <= N, n_w >= 1, non-NULL device pointers, even ld_w >= 2 n_w)");
        return LO_EINVAL;
    }
    const unsigned long long need = 16ull * (unsigned long long)n_w * (unsigned long long)n_occ * (unsigned long long)n_occ;
    if (need > LO_NOALLOC_SCRATCH_BYTES) {
        lo::set_error("lo_theta_noalloc: the overlap matrices need " + std::to_string(need) + " bytes of scratch (16 n_w n_occ^2), the static array holds " +
                      std::to_string((unsigned long long)LO_NOALLOC_SCRATCH_BYTES) + ": split the batch");
        return LO_EINVAL;
    }
    if (device < 0 || device >= NOALLOC_MAX_DEVICES || !g_noalloc_ptr[device]) {
        lo_status st = lo_theta_noalloc_init(device);       // first use on this device (call it yourself before a stream capture)
        if (st != LO_OK) return st;
    }
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) { lo::set_error(std::string("lo_theta_noalloc: cudaSetDevice: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    // the S1 launcher of the ordinary path wants a factor set for N, N_pad and its timers: a blank one on the stack (no device
    // state, timing off); scratch = the static array, output = the caller's panels
    lo_factors blank;
    blank.N = N;
    blank.N_pad = (N + lo::KTILE - 1) / lo::KTILE * lo::KTILE;
    lo::launch_s1(&blank, n_w, psi_dev, n_occ, n_occ, phi_dev, g_noalloc_ptr[device], status_dev, thetaT_dev, 0, ld_w, static_cast<cudaStream_t>(stream));
    e = cudaGetLastError();
    if (e != cudaSuccess) { lo::set_error(std::string("lo_theta_noalloc: kernel launch failed: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}
