// lo_oracle.cpp -- CPU ORACLE for the LO-AFQMC local energy.  TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Plain, slow, obviously-correct fp64 / std::complex<double> loops written from the paper
// (arxiv 2202.00832, /root/reference/PAPER.md).  It shares no code, header, table or helper with the
// CUDA path (paper_2202_00832_b200/csrc) and must only be imported / linked / executed by tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
//
// Notation: N basis functions (paper: M), O occupied orbitals per spin
// (paper: N), X Cholesky vectors (paper: X, index alpha; here g), Psi trial (paper: Phi_T, real in
// every config), Phi walker, Theta = Phi (Psi^T Phi)^-1 (paper: Q, Eq. 15).
// Array layouts (all row-major, C order):  h[N][N], L[X][N][N], psi[N][O], phi[N][O] (complex),
// theta[N][O] (complex), Lbar[X][O][N] (Lbar[g][i][p] = sum_q L[g][p][q] psi[q][i]), hbar[O][N],
// G[N][N] (G[p][q], Eq. 14), factors of pair (i<=j): U[r][N] (row K = left singular vector K over p),
// sigma[r], W[r][N] (row K = right singular vector K over q):  Y^{ij}_pq ~= sum_K U[K][p] sigma[K] W[K][q].
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): brute-force Eq. 10 = Eq. 16 = Eq. 17 = Eq. 19
// at T=0 on config 0; closed-form HF energy for Phi=Psi; occupied-rotation and walker-gauge invariance;
// Psi^T Theta = I, G^2 = G, tr G = O; N_occ=1 and N_chol=1 special cases; Eckart-Young; truncation bound;
// Jacobi SVD vs diagonal / rank-1 / Hilbert matrices and vs numpy.linalg.svd.
// The paper prints no numeric worked example of a local energy, so beyond those pins the energies
// are "parity unpinned" to any external number ("Oracle pins").
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;

namespace {

// ---- Theta = Phi (Psi^T Phi)^-1, Eq. 15, A = Psi^dagger Phi (Psi real).
// LU with partial pivoting, then the N row systems theta[p][:] A = phi[p][:].
// returns 0, or 1 when a pivot is zero / non-finite (singular overlap).
int theta_one(int N, int O, const double* psi, const cd* phi, cd* theta, cd* det_out) {
    std::vector<cd> A((size_t)O * O);
    for (int i = 0; i < O; ++i)
        for (int j = 0; j < O; ++j) {
            cd s = 0;
            for (int p = 0; p < N; ++p) s += psi[(size_t)p * O + i] * phi[(size_t)p * O + j];
            A[(size_t)i * O + j] = s;
        }
    // we need theta A = phi  <=>  A^T theta^T = phi^T : factor B = A^T = P^T L U
    std::vector<cd> B((size_t)O * O);
    for (int i = 0; i < O; ++i)
        for (int j = 0; j < O; ++j) B[(size_t)i * O + j] = A[(size_t)j * O + i];
    std::vector<int> piv(O);
    cd det = 1;
    for (int k = 0; k < O; ++k) {
        int r = k;
        double best = std::abs(B[(size_t)k * O + k]);
        for (int i = k + 1; i < O; ++i) {
            double v = std::abs(B[(size_t)i * O + k]);
            if (v > best) { best = v; r = i; }
        }
        if (!(best > 1e-300) || !std::isfinite(best)) return 1;
        piv[k] = r;
        if (r != k) {
            for (int j = 0; j < O; ++j) std::swap(B[(size_t)k * O + j], B[(size_t)r * O + j]);
            det = -det;
        }
        det *= B[(size_t)k * O + k];
        for (int i = k + 1; i < O; ++i) {
            cd f = B[(size_t)i * O + k] / B[(size_t)k * O + k];
            B[(size_t)i * O + k] = f;
            for (int j = k + 1; j < O; ++j) B[(size_t)i * O + j] -= f * B[(size_t)k * O + j];
        }
    }
    if (det_out) *det_out = det;
    std::vector<cd> x(O);
    for (int p = 0; p < N; ++p) {
        for (int i = 0; i < O; ++i) x[i] = phi[(size_t)p * O + i];
        for (int k = 0; k < O; ++k) std::swap(x[k], x[piv[k]]);
        for (int i = 0; i < O; ++i) {               // L y = P b (unit lower)
            cd s = x[i];
            for (int j = 0; j < i; ++j) s -= B[(size_t)i * O + j] * x[j];
            x[i] = s;
        }
        for (int i = O - 1; i >= 0; --i) {           // U t = y
            cd s = x[i];
            for (int j = i + 1; j < O; ++j) s -= B[(size_t)i * O + j] * x[j];
            x[i] = s / B[(size_t)i * O + i];
        }
        for (int i = 0; i < O; ++i) theta[(size_t)p * O + i] = x[i];
    }
    return 0;
}

// ---- one-sided (Hestenes) Jacobi SVD of a real n x n matrix, cyclic-by-rows sweeps.
// On exit: Ut[K][p] (row K = left vector), s[K] descending, Wt[K][q] (row K = right vector),
// A = sum_K Ut[K][:]^T s[K] Wt[K][:].  Columns whose norm is zero give s=0 and a zero left vector.
void jacobi_svd(int n, const double* A, double* Ut, double* s, double* Wt) {
    // work on columns: g[c][:] = column c of A (so g is A^T stored row-major), v = identity
    std::vector<double> g((size_t)n * n), v((size_t)n * n, 0.0);
    for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) g[(size_t)c * n + r] = A[(size_t)r * n + c];
    for (int c = 0; c < n; ++c) v[(size_t)c * n + c] = 1.0;
    const double tol = 1e-15;
    double fro2 = 0;
    for (size_t k = 0; k < (size_t)n * n; ++k) fro2 += A[k] * A[k];
    const double tiny2 = fro2 * 1e-30;              // columns below 1e-15 ||A||_F are numerically zero: left alone
    for (int sweep = 0; sweep < 60; ++sweep) {
        int rotations = 0;
        for (int p = 0; p < n - 1; ++p)
            for (int q = p + 1; q < n; ++q) {
                double* gp = &g[(size_t)p * n];
                double* gq = &g[(size_t)q * n];
                double a = 0, b = 0, c = 0;
                for (int k = 0; k < n; ++k) { a += gp[k] * gp[k]; b += gq[k] * gq[k]; c += gp[k] * gq[k]; }
                if (a <= tiny2 || b <= tiny2) continue;
                if (std::fabs(c) <= tol * std::sqrt(a * b)) continue;
                ++rotations;
                double zeta = (b - a) / (2.0 * c);
                double t = (zeta >= 0 ? 1.0 : -1.0) / (std::fabs(zeta) + std::sqrt(1.0 + zeta * zeta));
                double cs = 1.0 / std::sqrt(1.0 + t * t), sn = cs * t;
                for (int k = 0; k < n; ++k) {
                    double x = gp[k], y = gq[k];
                    gp[k] = cs * x - sn * y;
                    gq[k] = sn * x + cs * y;
                }
                double* vp = &v[(size_t)p * n];
                double* vq = &v[(size_t)q * n];
                for (int k = 0; k < n; ++k) {
                    double x = vp[k], y = vq[k];
                    vp[k] = cs * x - sn * y;
                    vq[k] = sn * x + cs * y;
                }
            }
        if (rotations == 0) break;
    }
    std::vector<double> nrm(n);
    for (int c = 0; c < n; ++c) {
        double a = 0;
        for (int k = 0; k < n; ++k) a += g[(size_t)c * n + k] * g[(size_t)c * n + k];
        nrm[c] = std::sqrt(a);
    }
    std::vector<int> order(n);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return nrm[x] > nrm[y]; });
    for (int K = 0; K < n; ++K) {
        int c = order[K];
        s[K] = nrm[c];
        for (int k = 0; k < n; ++k) {
            Ut[(size_t)K * n + k] = nrm[c] > 0 ? g[(size_t)c * n + k] / nrm[c] : 0.0;
            Wt[(size_t)K * n + k] = v[(size_t)c * n + k];
        }
    }
}

// Y^{ij}_pq = sum_g Lbar[g][i][p] Lbar[g][j][q]   (Y_ijrs)
void pair_eri(int N, int X, int O, const double* Lbar, int i, int j, double* Y) {
    std::fill(Y, Y + (size_t)N * N, 0.0);
    for (int g = 0; g < X; ++g) {
        const double* li = Lbar + ((size_t)g * O + i) * N;
        const double* lj = Lbar + ((size_t)g * O + j) * N;
        for (int p = 0; p < N; ++p) {
            double a = li[p];
            double* y = Y + (size_t)p * N;
            for (int q = 0; q < N; ++q) y[q] += a * lj[q];
        }
    }
}

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Eq. 15.  status: 0 ok, 1 singular overlap.  det (optional) = det(Psi^T Phi) = <Psi|Phi>.
int orc_theta(int N, int O, const double* psi, const cd* phi, cd* theta, cd* det) {
    return theta_one(N, O, psi, phi, theta, det);
}

// Eq. 14 with the index reading of SURVEY 8c-D2: G[p][q] = sum_i Theta[q][i] conj(Psi[p][i]) (Psi real).
void orc_green(int N, int O, const double* psi, const cd* theta, cd* G) {
    for (int p = 0; p < N; ++p)
        for (int q = 0; q < N; ++q) {
            cd s = 0;
            for (int i = 0; i < O; ++i) s += theta[(size_t)q * O + i] * psi[(size_t)p * O + i];
            G[(size_t)p * N + q] = s;
        }
}

// O1 -- brute-force definition.  Eq. 8 one-body + Eq. 10 with V_pqrs = sum_g L^g_pr L^g_qs
// and the spin sums written out for G^alpha, G^beta (closed shell: Ga == Gb):
//   E1  = sum_s sum_pq h_pq G^s_pq
//   E_J = 1/2 sum_pqrs V_pqrs (Ga+Gb)_pr (Ga+Gb)_qs
//   E_K = -1/2 sum_pqrs V_pqrs (Ga_ps Ga_qr + Gb_ps Gb_qr)
// out = {E1, E_J, E_K}.  Cost N^4 (+ X N^4 to build V): tiny inputs only.
void orc_energy_bruteforce(int N, int X, const double* h, const double* L, const cd* Ga, const cd* Gb, cd* out) {
    size_t N2 = (size_t)N * N;
    std::vector<double> V(N2 * N2, 0.0);            // V[p][q][r][s]
    for (int g = 0; g < X; ++g) {
        const double* Lg = L + (size_t)g * N2;
        for (int p = 0; p < N; ++p)
            for (int q = 0; q < N; ++q)
                for (int r = 0; r < N; ++r) {
                    double a = Lg[(size_t)p * N + r];
                    double* v = &V[(((size_t)p * N + q) * N + r) * N];
                    const double* lq = Lg + (size_t)q * N;
                    for (int s = 0; s < N; ++s) v[s] += a * lq[s];
                }
    }
    cd e1 = 0, ej = 0, ek = 0;
    for (int p = 0; p < N; ++p)
        for (int q = 0; q < N; ++q) e1 += h[(size_t)p * N + q] * (Ga[(size_t)p * N + q] + Gb[(size_t)p * N + q]);
    for (int p = 0; p < N; ++p)
        for (int q = 0; q < N; ++q)
            for (int r = 0; r < N; ++r)
                for (int s = 0; s < N; ++s) {
                    double v = V[(((size_t)p * N + q) * N + r) * N + s];
                    cd gpr = Ga[(size_t)p * N + r] + Gb[(size_t)p * N + r];
                    cd gqs = Ga[(size_t)q * N + s] + Gb[(size_t)q * N + s];
                    ej += 0.5 * v * gpr * gqs;
                    ek -= 0.5 * v * (Ga[(size_t)p * N + s] * Ga[(size_t)q * N + r] + Gb[(size_t)p * N + s] * Gb[(size_t)q * N + r]);
                }
    out[0] = e1; out[1] = ej; out[2] = ek;
}

// Half-rotated Cholesky vectors: Lbar[g][i][p] = sum_q L[g][p][q] psi[q][i]; hbar[i][p] = sum_q psi[q][i] h[q][p].
void orc_half_rotate(int N, int X, int O, const double* L, const double* h, const double* psi, double* Lbar, double* hbar) {
#pragma omp parallel for schedule(static)
    for (int g = 0; g < X; ++g)
        for (int i = 0; i < O; ++i)
            for (int p = 0; p < N; ++p) {
                double s = 0;
                for (int q = 0; q < N; ++q) s += L[((size_t)g * N + p) * N + q] * psi[(size_t)q * O + i];
                Lbar[((size_t)g * O + i) * N + p] = s;
            }
    for (int i = 0; i < O; ++i)
        for (int p = 0; p < N; ++p) {
            double s = 0;
            for (int q = 0; q < N; ++q) s += psi[(size_t)q * O + i] * h[(size_t)q * N + p];
            hbar[(size_t)i * N + p] = s;
        }
}

// One-body and Coulomb by the Cholesky route (Eq. 16 Coulomb part).
// n_spin = 1: E1 = 2 sum h̄Θ, E_J = 2 sum_g (X^g)^2;  n_spin = 2: E1 = sum_s sum h̄Θ, E_J = 1/2 sum_g (X_a+X_b)^2.
// Complex square, not modulus.  Xg (optional, [X]) receives sum_s X^g_s.  out = {E1, E_J}.
void orc_onebody_coulomb(int N, int X, int n_spin, const int* O, const double* const* Lbar, const double* const* hbar,
                         const cd* const* theta, cd* out, cd* Xg) {
    cd e1 = 0;
    for (int s = 0; s < n_spin; ++s)
        for (int i = 0; i < O[s]; ++i)
            for (int p = 0; p < N; ++p) e1 += hbar[s][(size_t)i * N + p] * theta[s][(size_t)p * O[s] + i];
    cd ej = 0;
    for (int g = 0; g < X; ++g) {
        cd x = 0;
        for (int s = 0; s < n_spin; ++s)
            for (int i = 0; i < O[s]; ++i)
                for (int p = 0; p < N; ++p) x += Lbar[s][((size_t)g * O[s] + i) * N + p] * theta[s][(size_t)p * O[s] + i];
        if (Xg) Xg[g] = x;
        ej += x * x;
    }
    if (n_spin == 1) { out[0] = 2.0 * e1; out[1] = 2.0 * ej; }
    else { out[0] = e1; out[1] = 0.5 * ej; }
}

// O2 -- exact exchange by the Cholesky route (Eq. 16 exchange part): T^g_ij = sum_p Lbar[g][i][p] Theta[p][j],
// E_K(spin) = - sum_g sum_ij T_ij T_ji.  Returns the single-spin sum (closed shell: E_K = this; unrestricted: 1/2 sum_s).
void orc_exchange_cholesky(int N, int X, int O, const double* Lbar, const cd* theta, cd* out) {
    cd ek = 0;
    std::vector<cd> T((size_t)O * O);
    for (int g = 0; g < X; ++g) {
        for (int i = 0; i < O; ++i)
            for (int j = 0; j < O; ++j) {
                cd s = 0;
                for (int p = 0; p < N; ++p) s += Lbar[((size_t)g * O + i) * N + p] * theta[(size_t)p * O + j];
                T[(size_t)i * O + j] = s;
            }
        for (int i = 0; i < O; ++i)
            for (int j = 0; j < O; ++j) ek -= T[(size_t)i * O + j] * T[(size_t)j * O + i];
    }
    *out = ek;
}

// Y^{ij} block of the half-rotated ERI tensor.
void orc_pair_eri(int N, int X, int O, const double* Lbar, int i, int j, double* Y) { pair_eri(N, X, O, Lbar, i, j, Y); }

// O3 -- exact exchange from the full pair ERIs (Eq. 17 exchange part): for i<=j,
// E_K -= m_ij sum_pq Y^{ij}_pq Theta_qi Theta_pj, m = 1 (i==j) or 2 (i<j) because Y^{ji} = (Y^{ij})^T.
// Blocks are formed on the fly.  Single-spin sum (see orc_exchange_cholesky).
void orc_exchange_full_eri(int N, int X, int O, const double* Lbar, const cd* theta, cd* out) {
    cd ek = 0;
    std::vector<double> Y((size_t)N * N);
    for (int i = 0; i < O; ++i)
        for (int j = i; j < O; ++j) {
            pair_eri(N, X, O, Lbar, i, j, Y.data());
            cd s = 0;
            for (int p = 0; p < N; ++p)
                for (int q = 0; q < N; ++q) s += Y[(size_t)p * N + q] * theta[(size_t)q * O + i] * theta[(size_t)p * O + j];
            ek -= (i == j ? 1.0 : 2.0) * s;
        }
    *out = ek;
}

// Jacobi SVD of an n x n matrix (rows of Ut/Wt are singular vectors, s descending).
void orc_svd(int n, const double* A, double* Ut, double* s, double* Wt) { jacobi_svd(n, A, Ut, s, Wt); }

// O4 -- own factor set (Eq. 18): full sorted SVD of the listed pair blocks; the caller keeps
// the leading r = #{sigma_K > T} rows (strict, absolute threshold).  OpenMP over pairs.
// Ut, Wt: [n_pairs][N][N], s: [n_pairs][N].
void orc_factor_pairs(int N, int X, int O, const double* Lbar, int n_pairs, const int* pi, const int* pj,
                      double* Ut, double* s, double* Wt) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_pairs; ++k) {
        std::vector<double> Y((size_t)N * N);
        pair_eri(N, X, O, Lbar, pi[k], pj[k], Y.data());
        jacobi_svd(N, Y.data(), Ut + (size_t)k * N * N, s + (size_t)k * N, Wt + (size_t)k * N * N);
    }
}

// O5 -- truncated exchange from a factor set (Eq. 19 / 22 exchange part):
// a_K = sum_p U[K][p] Theta[p][j], b_K = sum_q W[K][q] Theta[q][i], E_K(spin) = - sum_{i<=j} m_ij sum_K sigma_K a_K b_K.
// Factor set of one spin: pairs (pi[k], pj[k]) with rank r[k], rows stored back to back at row offset off[k]
// in U[.][N], sigma[.], W[.][N].  Single-spin sum.
void orc_exchange_lo(int N, int O, int n_pairs, const int* pi, const int* pj, const int* r, const int64_t* off,
                     const double* U, const double* sigma, const double* W, const cd* theta, cd* out) {
    cd ek = 0;
    for (int k = 0; k < n_pairs; ++k) {
        int i = pi[k], j = pj[k];
        cd e = 0;
        for (int K = 0; K < r[k]; ++K) {
            const double* u = U + (size_t)(off[k] + K) * N;
            const double* w = W + (size_t)(off[k] + K) * N;
            cd a = 0, b = 0;
            for (int p = 0; p < N; ++p) a += u[p] * theta[(size_t)p * O + j];
            for (int q = 0; q < N; ++q) b += w[q] * theta[(size_t)q * O + i];
            e += sigma[off[k] + K] * a * b;
        }
        ek -= (i == j ? 1.0 : 2.0) * e;
    }
    *out = ek;
}

// O5 for several walkers at once (the same sum as orc_exchange_lo, one walker per OpenMP task): thetas [n_w][N][O],
// out [n_w] single-spin sums.  Lets a checker stream a large factor set through in chunks of pairs and add up.
void orc_exchange_lo_batch(int n_w, int N, int O, int n_pairs, const int* pi, const int* pj, const int* r, const int64_t* off,
                           const double* U, const double* sigma, const double* W, const cd* thetas, cd* out) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int w = 0; w < n_w; ++w)
        orc_exchange_lo(N, O, n_pairs, pi, pj, r, off, U, sigma, W, thetas + (size_t)w * N * O, out + w);
}

// Paper-literal compressed Coulomb term (Eq. 19 / 22, "4 Q̄_{K,L,i} Q̄_{K,R,j}"):
// closed shell E_J^{LO} = 2 sum_{ij ordered} sum_K sigma_K (U^T Theta_i)_K (W Theta_j)_K, where the (j,i) block of an
// i<j pair, Y^{ji} = (Y^{ij})^T, contributes the same number as the (i,j) block (weight m_ij).  Returns the single-spin double sum S so that
// closed shell E_J^{LO} = 2 S.  Listed as NEXT-3 in SURVEY 8(f); exposed so the difference to the Cholesky route
// is documented.
void orc_coulomb_lo(int N, int O, int n_pairs, const int* pi, const int* pj, const int* r, const int64_t* off,
                    const double* U, const double* sigma, const double* W, const cd* theta, cd* out) {
    cd S = 0;
    for (int k = 0; k < n_pairs; ++k) {
        int i = pi[k], j = pj[k];
        cd e = 0;
        for (int K = 0; K < r[k]; ++K) {
            const double* u = U + (size_t)(off[k] + K) * N;
            const double* w = W + (size_t)(off[k] + K) * N;
            cd ui = 0, wj = 0;
            for (int p = 0; p < N; ++p) {
                ui += u[p] * theta[(size_t)p * O + i];
                wj += w[p] * theta[(size_t)p * O + j];
            }
            e += sigma[off[k] + K] * ui * wj;          // block (i,j); block (j,i) gives the same number:
        }                                              // sum_rs Y^{ji}_rs Q_rj Q_si = sum_rs Y^{ij}_sr Q_rj Q_si
        S += (i == j ? 1.0 : 2.0) * e;
    }
    *out = S;
}

// The whole LO local energy for a batch of walkers (steps S1-S5 of SURVEY 8(a) in the oracle's plain form):
// per walker Theta (Eq. 15), E1 and E_J by the Cholesky route, E_K from the given factor set (O5), E_L = E1+E_J+E_K.
// n_spin = 2 applies the unrestricted weights of SURVEY 8c-O6 (E_K = -1/2 sum_s ...).  OpenMP over walkers.
// phi[s]: [n_w][N][O_s].  out: [n_w][4] = {E_L, E1, E_J, E_K};  status[n_w] (0 ok, 1 singular -> NaN).
// This is the function bench.py times as "cpu_baseline".
void orc_local_energy_lo(int n_w, int N, int X, int n_spin, const int* O, const double* const* psi,
                         const double* const* Lbar, const double* const* hbar,
                         const int* n_pairs, const int* const* pi, const int* const* pj, const int* const* r,
                         const int64_t* const* off, const double* const* U, const double* const* sigma,
                         const double* const* W, const cd* const* phi, cd* out, int* status) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int w = 0; w < n_w; ++w) {
        std::vector<cd> th[2];
        const cd* thp[2] = {nullptr, nullptr};
        int bad = 0;
        for (int s = 0; s < n_spin; ++s) {
            th[s].resize((size_t)N * O[s]);
            bad |= theta_one(N, O[s], psi[s], phi[s] + (size_t)w * N * O[s], th[s].data(), nullptr);
            thp[s] = th[s].data();
        }
        cd* o = out + (size_t)w * 4;
        if (status) status[w] = bad;
        if (bad) {
            double nan = std::nan("");
            o[0] = o[1] = o[2] = o[3] = cd(nan, nan);
            continue;
        }
        cd e[2];
        orc_onebody_coulomb(N, X, n_spin, O, Lbar, hbar, thp, e, nullptr);
        cd ek = 0;
        for (int s = 0; s < n_spin; ++s) {
            cd t;
            orc_exchange_lo(N, O[s], n_pairs[s], pi[s], pj[s], r[s], off[s], U[s], sigma[s], W[s], thp[s], &t);
            ek += t;
        }
        if (n_spin == 2) ek *= 0.5;
        o[1] = e[0]; o[2] = e[1]; o[3] = ek; o[0] = e[0] + e[1] + ek;
    }
}

// NEXT-1 -- propagator formation ("forming the propagation matrix (B = sum_alpha x_alpha L_alpha),
// scaling as X M^2"): B[p][q] = sum_g x[g] L[g][p][q], x complex (shifted auxiliary fields), L real.
void orc_propagator(int N, int X, const double* L, const cd* x, cd* B) {
    for (int p = 0; p < N; ++p)
        for (int q = 0; q < N; ++q) {
            cd s = 0;
            for (int g = 0; g < X; ++g) s += x[g] * L[((size_t)g * N + p) * N + q];
            B[(size_t)p * N + q] = s;
        }
}

}  // extern "C"
