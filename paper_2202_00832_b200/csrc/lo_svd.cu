// lo_svd.cu -- the pair-block SVD of lo_setup (Eq. 18: "a list of N_cas x N_cas SVD decompositions"),
// host and device versions of ONE algorithm written for this library: a BLOCK one-sided Jacobi method with Gram
// subproblems.
//
//   The n rows g_c of G (row c = column c of Y^{ij}, so G = Y^T) are cut into blocks of SVD_B = 16 rows.  One sweep visits
//   every pair of blocks (I, J) once in a round-robin schedule ("chair rotation": the pairs of a round are disjoint, so a
//   round's subproblems are independent).  For a block pair the 32 x 32 Gram matrix S = A A^T of its rows A = [G_I; G_J]
//   is formed (a rank-n update: DMMA on the device), diagonalised S = Q diag(l) Q^T by a cyclic two-sided Jacobi
//   eigen-iteration on the small matrix, the eigenvectors are ordered by decreasing eigenvalue (longer rows drift to the
//   front, which takes 14 -> 10 sweeps at n = 378), and the rows are replaced by Q^T A (a 32 x 32 x n GEMM), V_I, V_J likewise.  A
//   block pair whose Gram matrix is already diagonal to working accuracy is left alone; the method stops after a sweep
//   in which every block pair was left alone.  Then sigma_K = |g_K|, U row K = g_K / sigma_K, W row K = v_K.
//
//   Working accuracy: a pair of rows (p, q) counts as orthogonal when |S_pq| <= tau sqrt(S_pp S_qq), tau = n u,
//   u = 2^-53 (the rounding level of an n-term dot product).  Rows with |g|^2 <= (n u)^2 |Y|_F^2 / n are numerically
//   null: whatever direction they have is rounding noise of earlier updates; they take no part in any rotation.
//
//   Every matrix reports the number of sweeps it took and the largest |S_pq| / sqrt(S_pp S_qq) seen in its last sweep
//   (lo_info: svd_sweeps_max, svd_offdiag_max); lo_setup fails with LO_EINTERNAL if SVD_MAX_SWEEPS did not suffice.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "lo_device.cuh"

namespace lo {

// Round-robin schedule over m = 2 * half blocks by chair rotation: block m-1 keeps its chair, the others move one chair on
// after every round.  sched[(round * half + k) * 2 + {0,1}] = the two blocks of subproblem k in that round; m - 1 rounds.
std::vector<int> svd_schedule(int n_blocks) {
    const int m = std::max(2, n_blocks + (n_blocks & 1)), half = m / 2;
    std::vector<int> chair(m);
    std::iota(chair.begin(), chair.end(), 0);
    std::vector<int> sched;
    sched.reserve((size_t)(m - 1) * half * 2);
    for (int round = 0; round < m - 1; ++round) {
        for (int k = 0; k < half; ++k) {
            int a = chair[k], b = chair[m - 1 - k];
            if (a > b) std::swap(a, b);
            sched.push_back(a);
            sched.push_back(b);          // b >= n_blocks marks the dummy block of an odd count
        }
        std::rotate(chair.begin(), chair.begin() + 1, chair.begin() + (m - 1));
    }
    return sched;
}

namespace {

constexpr double SVD_U = 1.1102230246251565e-16;   // unit roundoff 2^-53

// Rotation that diagonalises [[app, apq], [apq, aqq]]: new_p = c x_p + s x_q, new_q = -s x_p + c x_q, with the angle of
// smaller magnitude (|phi| <= pi/4), from the half-angle identities: cos 2phi = |d| / h, sin 2phi = sgn(d) o / h,
// d = app - aqq, o = 2 apq, h = hypot(d, o).
inline void plane_angle(double app, double aqq, double apq, double& c, double& s) {
    const double d = app - aqq, o = 2.0 * apq, h = std::hypot(d, o);
    const double c2 = std::fabs(d) / h;
    c = std::sqrt(0.5 * (1.0 + c2));
    s = (d < 0.0 ? -o : o) / (2.0 * h * c);
}

// Cyclic two-sided Jacobi on the symmetric m x m matrix S (leading dimension ld); Q (m x m, ld) accumulates the rotations
// (columns = eigenvectors: S_in = Q diag Q^T).  Rows/columns with live[c] == false are left untouched.
void sym_jacobi_host(int m, double* S, double* Q, int ld, const bool* live, double tau) {
    for (int r = 0; r < m; ++r)
        for (int c = 0; c < m; ++c) Q[r * ld + c] = r == c ? 1.0 : 0.0;
    for (int it = 0; it < 40; ++it) {
        bool rotated = false;
        for (int p = 0; p < m - 1; ++p)
            for (int q = p + 1; q < m; ++q) {
                if (!live[p] || !live[q]) continue;
                const double apq = S[p * ld + q], app = S[p * ld + p], aqq = S[q * ld + q];
                if (std::fabs(apq) <= tau * std::sqrt(app * aqq)) continue;
                rotated = true;
                double c, s;
                plane_angle(app, aqq, apq, c, s);
                for (int k = 0; k < m; ++k) {      // columns p, q of S and of Q
                    const double x = S[k * ld + p], y = S[k * ld + q];
                    S[k * ld + p] = c * x + s * y;
                    S[k * ld + q] = c * y - s * x;
                    const double qx = Q[k * ld + p], qy = Q[k * ld + q];
                    Q[k * ld + p] = c * qx + s * qy;
                    Q[k * ld + q] = c * qy - s * qx;
                }
                for (int k = 0; k < m; ++k) {      // rows p, q of S
                    const double x = S[p * ld + k], y = S[q * ld + k];
                    S[p * ld + k] = c * x + s * y;
                    S[q * ld + k] = c * y - s * x;
                }
                S[p * ld + q] = S[q * ld + p] = 0.0;
            }
        if (!rotated) break;
    }
}

}  // namespace

// Host version.  G: R rows of length len (for a pair block: R = len = N, row c = column c of Y), overwritten by the
// orthogonalised rows; V (R x R, may be NULL) receives the accumulated transformation.  sigma: the row lengths,
// descending; order[K] = row of G / V that holds singular triplet K.
void host_block_svd(int R, int len, double* G, double* V, std::vector<double>& sigma, std::vector<int>& order, double skip_below, SvdStat* stat) {
    const int B = SVD_B, nb = (R + B - 1) / B, M = 2 * B, dim = std::max(R, len);
    if (V) {
        std::fill(V, V + (size_t)R * R, 0.0);
        for (int c = 0; c < R; ++c) V[(size_t)c * R + c] = 1.0;
    }
    double fro2 = 0;
    for (size_t k = 0; k < (size_t)R * len; ++k) fro2 += G[k] * G[k];
    if (std::sqrt(fro2) * (1.0 + 1e-12) <= skip_below) {
        // sigma_1 <= |Y|_F <= threshold: rank 0 whatever the vectors are (second level of the pair screen); sigma_1 is
        // reported as its bound |Y|_F
        sigma.assign(R, 0.0);
        sigma[0] = std::sqrt(fro2) * (1.0 + 1e-12);
        order.resize(R);
        std::iota(order.begin(), order.end(), 0);
        if (stat) { stat->sweeps = 0; stat->offdiag = 0; stat->converged = true; stat->screened = 1; }
        return;
    }
    const double tau = dim * SVD_U, null2 = tau * tau * fro2 / dim;
    const std::vector<int> sched = svd_schedule(nb);
    const int half = std::max(2, nb + (nb & 1)) / 2, rounds = 2 * half - 1;
    std::vector<double> S((size_t)M * M), Q((size_t)M * M), Qs, tmp((size_t)M * std::max(len, R));
    int rows[2 * SVD_B];
    bool live[2 * SVD_B];
    int sweep = 0;
    double worst = 0;
    for (; sweep < SVD_MAX_SWEEPS; ++sweep) {
        bool touched = false;
        worst = 0;
        for (int round = 0; round < rounds; ++round)
            for (int k = 0; k < half; ++k) {
                const int bI = sched[((size_t)round * half + k) * 2], bJ = sched[((size_t)round * half + k) * 2 + 1];
                int m = 0;
                for (int blk : {bI, bJ})
                    for (int c = blk * B; c < std::min(R, (blk + 1) * B); ++c)
                        if (blk < nb) rows[m++] = c;
                if (m < 2) continue;
                for (int a = 0; a < m; ++a)
                    for (int b = a; b < m; ++b) {
                        const double *x = G + (size_t)rows[a] * len, *y = G + (size_t)rows[b] * len;
                        double acc = 0;
                        for (int e = 0; e < len; ++e) acc += x[e] * y[e];
                        S[a * M + b] = S[b * M + a] = acc;
                    }
                double off = 0;
                for (int a = 0; a < m; ++a) live[a] = S[a * M + a] > null2;
                for (int a = 0; a < m; ++a)
                    for (int b = a + 1; b < m; ++b)
                        if (live[a] && live[b]) off = std::max(off, std::fabs(S[a * M + b]) / std::sqrt(S[a * M + a] * S[b * M + b]));
                worst = std::max(worst, off);
                if (off <= tau) continue;
                touched = true;
                sym_jacobi_host(m, S.data(), Q.data(), M, live, 0.25 * tau);
                {   // the new rows take the places of the old live rows in order of decreasing length (= diagonal of S)
                    int from[2 * SVD_B], place[2 * SVD_B], nl = 0;
                    for (int a = 0; a < m; ++a)
                        if (live[a]) { from[nl] = a; place[nl] = a; ++nl; }
                    std::stable_sort(from, from + nl, [&](int x, int y) { return S[x * M + x] > S[y * M + y]; });
                    Qs = Q;
                    for (int t = 0; t < nl; ++t)
                        for (int b = 0; b < m; ++b) Q[b * M + place[t]] = Qs[b * M + from[t]];
                }
                for (int pass = 0; pass < (V ? 2 : 1); ++pass) {          // rows <- Q^T rows
                    double* X = pass == 0 ? G : V;
                    const int w = pass == 0 ? len : R;
                    for (int a = 0; a < m; ++a) {
                        double* t = tmp.data() + (size_t)a * w;
                        std::fill(t, t + w, 0.0);
                        for (int b = 0; b < m; ++b) {
                            const double q = Q[b * M + a];
                            if (q == 0.0) continue;
                            const double* x = X + (size_t)rows[b] * w;
                            for (int e = 0; e < w; ++e) t[e] += q * x[e];
                        }
                    }
                    for (int a = 0; a < m; ++a) std::memcpy(X + (size_t)rows[a] * w, tmp.data() + (size_t)a * w, (size_t)w * 8);
                }
            }
        if (!touched) break;
    }
    if (stat) { stat->sweeps = sweep; stat->offdiag = worst; stat->converged = sweep < SVD_MAX_SWEEPS; }
    std::vector<double> rl(R);
    for (int c = 0; c < R; ++c) {
        double a = 0;
        for (int e = 0; e < len; ++e) a += G[(size_t)c * len + e] * G[(size_t)c * len + e];
        rl[c] = std::sqrt(a);
    }
    order.resize(R);
    std::iota(order.begin(), order.end(), 0);
    std::sort(order.begin(), order.end(), [&](int x, int y) { return rl[x] != rl[y] ? rl[x] > rl[y] : x < y; });
    sigma.resize(R);
    for (int K = 0; K < R; ++K) sigma[K] = rl[order[K]];
}

// Host version of the randomised SVD of one pair block (steps as in gpu_pair_rsvd, lo_setup_gpu.cu): G = Y^T, N x N.
bool host_pair_rsvd(int N, int k, const double* G, std::vector<double>& sigma, std::vector<double>& U, std::vector<double>& W, SvdStat* stat) {
    std::vector<double> Zt((size_t)k * N, 0.0), Bp((size_t)k * N, 0.0), Vr((size_t)k * k), sg;
    std::vector<int> order;
    const unsigned long long seed = 0x2202008320000000ull + (unsigned long long)k;
    for (int q = 0; q < N; ++q)                                   // Zt[kk][q] = sum_p Om[p][kk] G[q][p]
        for (int p = 0; p < N; ++p) {
            const double g = G[(size_t)q * N + p];
            for (int kk = 0; kk < k; ++kk) Zt[(size_t)kk * N + q] += gauss_at(seed, (unsigned long long)p * k + kk) * g;
        }
    SvdStat st1, st2;
    host_block_svd(k, N, Zt.data(), nullptr, sg, order, -1.0, &st1);
    for (int kk = 0; kk < k; ++kk) {                              // orthonormal rows; a null row (sketch wider than the rank) -> 0
        double a = 0;
        for (int q = 0; q < N; ++q) a += Zt[(size_t)kk * N + q] * Zt[(size_t)kk * N + q];
        const double tau = N * SVD_U, inv = a > tau * tau * sg[0] * sg[0] ? 1.0 / std::sqrt(a) : 0.0;
        for (int q = 0; q < N; ++q) Zt[(size_t)kk * N + q] *= inv;
    }
    for (int kk = 0; kk < k; ++kk)                                // Bp = Pt G
        for (int q = 0; q < N; ++q) {
            const double pz = Zt[(size_t)kk * N + q];
            if (pz == 0.0) continue;
            for (int c = 0; c < N; ++c) Bp[(size_t)kk * N + c] += pz * G[(size_t)q * N + c];
        }
    host_block_svd(k, N, Bp.data(), Vr.data(), sg, order, -1.0, &st2);
    std::vector<double> Wf((size_t)k * N, 0.0);                   // Wf = Vr Pt
    for (int K = 0; K < k; ++K)
        for (int kk = 0; kk < k; ++kk) {
            const double v = Vr[(size_t)K * k + kk];
            if (v == 0.0) continue;
            for (int q = 0; q < N; ++q) Wf[(size_t)K * N + q] += v * Zt[(size_t)kk * N + q];
        }
    double r2 = 0, s2 = 0;                                        // |G - Wf^T Bp|_F^2 and |Bp|_F^2
    for (int q = 0; q < N; ++q)
        for (int c = 0; c < N; ++c) {
            double acc = 0;
            for (int K = 0; K < k; ++K) acc += Wf[(size_t)K * N + q] * Bp[(size_t)K * N + c];
            const double d = G[(size_t)q * N + c] - acc;
            r2 += d * d;
        }
    for (double v : sg) s2 += v * v;
    if (stat) { stat->sweeps = std::max(st1.sweeps, st2.sweeps); stat->offdiag = std::max(st1.offdiag, st2.offdiag); stat->converged = true; }
    if (!st1.converged || !st2.converged || !(std::sqrt(r2) <= 16.0 * N * SVD_U * std::sqrt(s2 + r2))) return false;
    sigma = sg;
    U.assign((size_t)k * N, 0.0);
    W.assign((size_t)k * N, 0.0);
    for (int K = 0; K < k; ++K) {
        const int c = order[K];
        const double inv = sg[K] > 0 ? 1.0 / sg[K] : 0.0;
        for (int e = 0; e < N; ++e) {
            U[(size_t)K * N + e] = Bp[(size_t)c * N + e] * inv;
            W[(size_t)K * N + e] = Wf[(size_t)c * N + e];
        }
    }
    return true;
}

// =====================================================================================================================
// Device version: one CTA of SVD_WARPS warps per matrix; every warp owns whole block-pair subproblems of the current
// round (Gram by DMMA from global memory, eigen-iteration in its own shared-memory slice, Q^T application by DMMA in
// place); __syncthreads() separates the rounds.  G: [n rows][ld] row-major, V: [n][ldv] (or NULL: no accumulation), ld and
// ldv multiples of 8, padding columns zero.  For a pair block n = N and ld = ldv = N_pad; the randomised path also runs it
// on k x N_pad sketches (n = k rows).
// =====================================================================================================================
namespace {

constexpr int SVD_WARPS = 4;
constexpr int SVD_M = 2 * SVD_B;            // rows of a subproblem (32 = one per lane)
constexpr int SVD_LDS = SVD_M + 1;          // shared-memory leading dimension (conflict-free row and column walks)

__device__ __forceinline__ double wmax(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// S (32 x 32, symmetric, lds SVD_LDS) -> Q; one warp; rows with S_cc <= null2 are dead.  Round-robin over the 32 indices
// by the same chair rotation as the block schedule (16 disjoint index pairs per round, 31 rounds per inner sweep).
__device__ void sym_jacobi_warp(double* S, double* Q, double* cs, int* pq, double null2, double tau, int lane) {
    for (int r = 0; r < SVD_M; ++r) Q[r * SVD_LDS + lane] = r == lane ? 1.0 : 0.0;
    const bool alive = S[lane * SVD_LDS + lane] > null2;
    const unsigned live_mask = __ballot_sync(0xffffffffu, alive);
    __syncwarp();
    int chair = lane;                        // chair[k] of the rotation, one per lane
    for (int it = 0; it < 30; ++it) {
        bool any = false;
        for (int round = 0; round < SVD_M - 1; ++round) {
            // partner of chair k is chair 31 - k
            const int mine = chair, other = __shfl_sync(0xffffffffu, chair, SVD_M - 1 - lane);
            bool rot = false;
            if (lane < SVD_M / 2) {
                const int p = min(mine, other), q = max(mine, other);
                double c = 1.0, s = 0.0;
                if (((live_mask >> p) & 1u) && ((live_mask >> q) & 1u)) {
                    const double apq = S[p * SVD_LDS + q], app = S[p * SVD_LDS + p], aqq = S[q * SVD_LDS + q];
                    if (fabs(apq) > tau * sqrt(app * aqq)) {
                        const double d = app - aqq, o = 2.0 * apq, h = hypot(d, o);
                        const double c2 = fabs(d) / h;
                        c = sqrt(0.5 * (1.0 + c2));
                        s = (d < 0.0 ? -o : o) / (2.0 * h * c);
                        rot = true;
                    }
                }
                cs[2 * lane] = c;
                cs[2 * lane + 1] = s;
                pq[2 * lane] = p;
                pq[2 * lane + 1] = rot ? q : -1;
            }
            const bool round_rot = __any_sync(0xffffffffu, rot);
            __syncwarp();
            if (round_rot) {
                any = true;
                // columns p, q of S and Q: lane = row
#pragma unroll 4
                for (int k = 0; k < SVD_M / 2; ++k) {
                    const int q = pq[2 * k + 1];
                    if (q < 0) continue;
                    const int p = pq[2 * k];
                    const double c = cs[2 * k], s = cs[2 * k + 1];
                    const double x = S[lane * SVD_LDS + p], y = S[lane * SVD_LDS + q];
                    S[lane * SVD_LDS + p] = c * x + s * y;
                    S[lane * SVD_LDS + q] = c * y - s * x;
                    const double qx = Q[lane * SVD_LDS + p], qy = Q[lane * SVD_LDS + q];
                    Q[lane * SVD_LDS + p] = c * qx + s * qy;
                    Q[lane * SVD_LDS + q] = c * qy - s * qx;
                }
                __syncwarp();
                // rows p, q of S: lane = column
#pragma unroll 4
                for (int k = 0; k < SVD_M / 2; ++k) {
                    const int q = pq[2 * k + 1];
                    if (q < 0) continue;
                    const int p = pq[2 * k];
                    const double c = cs[2 * k], s = cs[2 * k + 1];
                    const double x = S[p * SVD_LDS + lane], y = S[q * SVD_LDS + lane];
                    S[p * SVD_LDS + lane] = (lane == q) ? 0.0 : c * x + s * y;
                    S[q * SVD_LDS + lane] = (lane == p) ? 0.0 : c * y - s * x;
                }
            }
            __syncwarp();
            // chair rotation: chairs 0..30 move on by one, chair 31 stays
            const int nxt = __shfl_sync(0xffffffffu, chair, (lane + 1) % (SVD_M - 1));
            if (lane < SVD_M - 1) chair = nxt;
        }
        if (!any) break;
    }
    __syncwarp();
}

__global__ void __launch_bounds__(SVD_WARPS * 32) k_block_jacobi(double* __restrict__ Gall, double* __restrict__ Vall, int n, int len, int ld, int ldv,
                                                                 const int* __restrict__ sched, int half, int max_sweeps, double skip_below,
                                                                 int* __restrict__ sweeps_out, double* __restrict__ off_out,
                                                                 const int* __restrict__ idx, size_t stride) {
    extern __shared__ double sm[];
    __shared__ int s_touched;
    __shared__ double s_red[SVD_WARPS];
    __shared__ double s_off[SVD_WARPS];
    const int x = idx ? idx[blockIdx.x] : blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    double* G = Gall + (size_t)x * stride;                        // matrix x (statistics go to slot x as well)
    double* V = Vall ? Vall + (size_t)x * stride : nullptr;       // n rows of ldv >= n columns (a multiple of 8), or no accumulation
    double* S = sm + (size_t)warp * (2 * SVD_M * SVD_LDS + 2 * SVD_M);
    double* Q = S + SVD_M * SVD_LDS;
    double* cs = Q + SVD_M * SVD_LDS;
    int* pq = reinterpret_cast<int*>(cs + SVD_M);
    // V = I, |Y|_F^2
    double fro = 0;
    for (size_t e = tid; e < (size_t)n * ld; e += SVD_WARPS * 32) {
        const double v = G[e];
        fro = fma(v, v, fro);
    }
    if (V)
        for (size_t e = tid; e < (size_t)n * ldv; e += SVD_WARPS * 32) V[e] = (e / ldv == e % ldv) ? 1.0 : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) fro += __shfl_xor_sync(0xffffffffu, fro, o);
    if (lane == 0) s_red[warp] = fro;
    __syncthreads();
    fro = 0;
    for (int w = 0; w < SVD_WARPS; ++w) fro += s_red[w];
    if (sqrt(fro) * (1.0 + 1e-12) <= skip_below) {       // |Y|_F <= threshold: rank 0, no iteration (sweeps = -1, off = the bound)
        if (tid == 0) { sweeps_out[x] = -1; off_out[x] = sqrt(fro) * (1.0 + 1e-12); }
        return;
    }
    const int dim = max(n, len);           // len = true row length (<= ld)
    const double tau = dim * SVD_U, null2 = tau * tau * fro / dim;
    const int rounds = 2 * half - 1, nb = (n + SVD_B - 1) / SVD_B;
    int sweep = 0;
    double worst_cta = 0;
    for (; sweep < max_sweeps; ++sweep) {
        if (tid == 0) s_touched = 0;
        double worst = 0;
        __syncthreads();
        for (int round = 0; round < rounds; ++round) {
            for (int k = warp; k < half; k += SVD_WARPS) {
                const int bI = sched[(round * half + k) * 2], bJ = sched[(round * half + k) * 2 + 1];
                // global row of subproblem row m: m < 16 -> block I, else block J; rows >= n (ragged / dummy block) are zero
                auto grow = [&](int m) { return (m < SVD_B ? bI : bJ) * SVD_B + (m & (SVD_B - 1)); };
                // ---- Gram S = A A^T on the DMMA pipe: 4 row tiles of 8; the A fragment of tile j is also the B fragment of column tile j
                int rowt[4];
                bool okt[4];
#pragma unroll
                for (int ti = 0; ti < 4; ++ti) { rowt[ti] = grow(ti * 8 + g); okt[ti] = rowt[ti] < n && (ti < 2 || bJ < nb); }
                double acc[10][2];
#pragma unroll
                for (int a = 0; a < 10; ++a) acc[a][0] = acc[a][1] = 0.0;
                // two column chunks of 8 ahead: the loads of chunks k0 + 8 and k0 + 16 are in flight under the MMAs of chunk k0
                double f[2][4], f1[2][4];
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2)
#pragma unroll
                    for (int ti = 0; ti < 4; ++ti) {
                        f[h2][ti] = okt[ti] ? G[(size_t)rowt[ti] * ld + 4 * h2 + t] : 0.0;
                        f1[h2][ti] = (okt[ti] && 8 < ld) ? G[(size_t)rowt[ti] * ld + 8 + 4 * h2 + t] : 0.0;
                    }
                for (int k0 = 0; k0 < ld; k0 += 8) {
                    double f2[2][4];
#pragma unroll
                    for (int h2 = 0; h2 < 2; ++h2)
#pragma unroll
                        for (int ti = 0; ti < 4; ++ti) f2[h2][ti] = (okt[ti] && k0 + 16 < ld) ? G[(size_t)rowt[ti] * ld + k0 + 16 + 4 * h2 + t] : 0.0;
#pragma unroll
                    for (int h2 = 0; h2 < 2; ++h2) {
                        int a = 0;
#pragma unroll
                        for (int ti = 0; ti < 4; ++ti)
#pragma unroll
                            for (int tj = ti; tj < 4; ++tj, ++a) mma884(acc[a][0], acc[a][1], f[h2][ti], f[h2][tj]);
                    }
#pragma unroll
                    for (int h2 = 0; h2 < 2; ++h2)
#pragma unroll
                        for (int ti = 0; ti < 4; ++ti) { f[h2][ti] = f1[h2][ti]; f1[h2][ti] = f2[h2][ti]; }
                }
                {
                    int a = 0;
#pragma unroll
                    for (int ti = 0; ti < 4; ++ti)
#pragma unroll
                        for (int tj = ti; tj < 4; ++tj, ++a) {
                            const int r = ti * 8 + g, c = tj * 8 + 2 * t;
                            S[r * SVD_LDS + c] = acc[a][0];
                            S[r * SVD_LDS + c + 1] = acc[a][1];
                            if (tj > ti) { S[c * SVD_LDS + r] = acc[a][0]; S[(c + 1) * SVD_LDS + r] = acc[a][1]; }
                        }
                }
                __syncwarp();
                // ---- is the subproblem already diagonal to working accuracy?  lane = row
                const double dl = S[lane * SVD_LDS + lane];
                double off = 0;
                if (dl > null2) {
                    for (int c = 0; c < SVD_M; ++c) {
                        const double dc = S[c * SVD_LDS + c];
                        if (c != lane && dc > null2) off = fmax(off, fabs(S[lane * SVD_LDS + c]) / sqrt(dl * dc));
                    }
                }
                off = wmax(off);
                worst = fmax(worst, off);
                if (off <= tau) continue;            // warp-uniform
                if (lane == 0) s_touched = 1;
                sym_jacobi_warp(S, Q, cs, pq, null2, 0.25 * tau, lane);
                // the new rows take the places of the old live rows in order of decreasing length (= diagonal of S):
                // column `lane` of Q moves to column dest; pq[c] = source column of new column c
                {
                    const double dn = S[lane * SVD_LDS + lane];
                    const bool alive = dl > null2;
                    const unsigned live_mask = __ballot_sync(0xffffffffu, alive);
                    int rank = 0;
                    for (int c = 0; c < SVD_M; ++c) {
                        const double dc = __shfl_sync(0xffffffffu, dn, c);
                        rank += (((live_mask >> c) & 1u) && (dc > dn || (dc == dn && c < lane))) ? 1 : 0;
                    }
                    const int dest = alive ? (int)__fns(live_mask, 0, rank + 1) : lane;
                    __syncwarp();
                    pq[dest] = lane;
                    __syncwarp();
                }
                // ---- rows <- Q^T rows for G and V, in place, 8 columns at a time:  D[m][c] = sum_k Q[k][m] X[row_k][c]
                double qa[4][8];                     // A fragments of Q^T: tile mt, k-step ks: Q[ks*4 + t][mt*8 + g]
#pragma unroll
                for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) qa[mt][ks] = Q[(ks * 4 + t) * SVD_LDS + pq[mt * 8 + g]];
                int rowk[8];
                bool okk[8];
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) { rowk[ks] = grow(ks * 4 + t); okk[ks] = rowk[ks] < n && (ks < 4 || bJ < nb); }
#pragma unroll 1
                for (int pass = 0; pass < (V ? 2 : 1); ++pass) {
                    double* X = pass == 0 ? G : V;
                    const int ldx = pass == 0 ? ld : ldv;
                    double bf[8], b1[8];
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        bf[ks] = okk[ks] ? X[(size_t)rowk[ks] * ldx + g] : 0.0;
                        b1[ks] = (okk[ks] && 8 < ldx) ? X[(size_t)rowk[ks] * ldx + 8 + g] : 0.0;
                    }
                    for (int c0 = 0; c0 < ldx; c0 += 8) {
                        double nx[8];
                        const int c1 = c0 + 16;
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks) nx[ks] = (c1 < ldx && okk[ks]) ? X[(size_t)rowk[ks] * ldx + c1 + g] : 0.0;
                        double d[4][2];
#pragma unroll
                        for (int mt = 0; mt < 4; ++mt) d[mt][0] = d[mt][1] = 0.0;
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks)
#pragma unroll
                            for (int mt = 0; mt < 4; ++mt) mma884(d[mt][0], d[mt][1], qa[mt][ks], bf[ks]);
                        __syncwarp();                // every lane's loads of this column chunk are done before any store
#pragma unroll
                        for (int mt = 0; mt < 4; ++mt)
                            if (okt[mt]) *reinterpret_cast<double2*>(&X[(size_t)rowt[mt] * ldx + c0 + 2 * t]) = make_double2(d[mt][0], d[mt][1]);
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks) { bf[ks] = b1[ks]; b1[ks] = nx[ks]; }
                    }
                }
            }
            __syncthreads();                         // the next round's subproblems read rows this round wrote
        }
        if (lane == 0) s_off[warp] = worst;
        __syncthreads();
        worst_cta = 0;
        for (int w = 0; w < SVD_WARPS; ++w) worst_cta = fmax(worst_cta, s_off[w]);
        const int touched = s_touched;
        __syncthreads();
        if (!touched) break;
    }
    if (tid == 0) { sweeps_out[x] = sweep; off_out[x] = worst_cta; }
}

}  // namespace

size_t svd_kernel_smem() { return (size_t)SVD_WARPS * (2 * SVD_M * SVD_LDS + 2 * SVD_M) * 8; }

// Batched device SVD driver step: orthogonalise the rows of n_mat matrices in G (V <- accumulated transformation); matrix
// m of the launch is slot x = dIdx[m] (or m) at G + x * stride, V + x * stride.  dSched: device copy of
// svd_schedule(ceil(n/16)); dSweeps[x], dOff[x] receive the statistics.
cudaError_t launch_block_jacobi(double* G, double* V, int n_mat, int n, int len, int ld, int ldv, const int* dSched, double skip_below, int* dSweeps,
                                double* dOff, const int* dIdx, size_t stride, cudaStream_t stream) {
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_block_jacobi, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)svd_kernel_smem());
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const int nb = (n + SVD_B - 1) / SVD_B, half = std::max(2, nb + (nb & 1)) / 2;
    k_block_jacobi<<<n_mat, SVD_WARPS * 32, svd_kernel_smem(), stream>>>(G, V, n, len, ld, ldv, dSched, half, SVD_MAX_SWEEPS, skip_below, dSweeps, dOff, dIdx, stride);
    return cudaGetLastError();
}

}  // namespace lo
