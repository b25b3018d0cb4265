// lo_setup_gpu.cu -- device side of lo_setup (flag LO_SETUP_GPU_SVD): pair blocks Y^{ij}, the epilogue of
// their SVDs (Eq. 18; the iteration itself is the block Jacobi method of lo_svd.cu) and the packing copies.
// Setup is untimed.
#include <algorithm>
#include <cmath>

#include "lo_internal.h"

namespace lo {
namespace {

// G_x[q][p] = sum_g Lbar[g][oj][q] * Lbar[g][oi][p]   (row q of G = column q of Y^{ij});  [n][N][N_pad], pad = 0.
// 64 x 64 tile per CTA, 16 x 16 threads, 4 x 4 micro-tile, K chunk 16 staged in shared memory.
__global__ void __launch_bounds__(256) k_pair_gram(const double* __restrict__ Lbar, int n_chol, int O_tot, int N, int N_pad, int o_base,
                                                   const int* __restrict__ pi, const int* __restrict__ pj, double* __restrict__ G) {
    __shared__ double As[16][64 + 4], Bs[16][64 + 4];
    const int x = blockIdx.z, q0 = blockIdx.y * 64, p0 = blockIdx.x * 64;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const size_t gs = (size_t)O_tot * N_pad;
    const double* Li = Lbar + (size_t)(o_base + pi[x]) * N_pad;
    const double* Lj = Lbar + (size_t)(o_base + pj[x]) * N_pad;
    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
    for (int g0 = 0; g0 < n_chol; g0 += 16) {
        __syncthreads();
        for (int e = threadIdx.x; e < 16 * 64; e += 256) {
            int kk = e >> 6, c = e & 63, g = g0 + kk;
            bool okg = g < n_chol;
            As[kk][c] = (okg && q0 + c < N_pad) ? Lj[(size_t)g * gs + q0 + c] : 0.0;
            Bs[kk][c] = (okg && p0 + c < N_pad) ? Li[(size_t)g * gs + p0 + c] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { a[u] = As[kk][ty * 4 + u]; b[u] = Bs[kk][tx * 4 + u]; }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int v = 0; v < 4; ++v) acc[u][v] = fma(a[u], b[v], acc[u][v]);
        }
    }
    double* Gx = G + (size_t)x * N * N_pad;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        int q = q0 + ty * 4 + u;
        if (q >= N) continue;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            int p = p0 + tx * 4 + v;
            if (p < N_pad) Gx[(size_t)q * N_pad + p] = (p < N) ? acc[u][v] : 0.0;
        }
    }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sigma_K = |g_{order[K]}| descending;  U row K = g/sigma;  W row K = v.  R rows per matrix (R = N for a full pair block,
// R = k for a sketch); matrix x = idx[blockIdx.x] (or blockIdx.x) reads G/V at x * in_stride and writes slot x of the
// [.][N][N_pad] outputs; sigma / order entries R..N-1 are set to 0 / -1.
__global__ void __launch_bounds__(512) k_svd_finish(const double* __restrict__ Gall, const double* __restrict__ Vall, size_t in_stride, int R,
                                                    int N, int N_pad, const int* __restrict__ idx, double* __restrict__ sigma,
                                                    int* __restrict__ order, double* __restrict__ Uall, double* __restrict__ Wall) {
    extern __shared__ double nrm[];   // [R]
    const int x = idx ? idx[blockIdx.x] : blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* G = Gall + (size_t)x * in_stride;
    const double* V = Vall + (size_t)x * in_stride;
    for (int c = warp; c < R; c += 16) {
        double a = 0;
        for (int e = lane; e < N; e += 32) { double g = G[(size_t)c * N_pad + e]; a = fma(g, g, a); }
        a = warp_sum(a);
        if (lane == 0) nrm[c] = sqrt(a);
    }
    __syncthreads();
    for (int c = tid; c < N; c += 512) {
        if (c >= R) { order[(size_t)x * N + c] = -1; sigma[(size_t)x * N + c] = 0.0; continue; }
        const double v = nrm[c];
        int rank = 0;
        for (int d = 0; d < R; ++d) {
            const double u = nrm[d];
            rank += (u > v) || (u == v && d < c);
        }
        order[(size_t)x * N + rank] = c;
        sigma[(size_t)x * N + rank] = v;
    }
    __syncthreads();
    __threadfence_block();
    double* U = Uall + (size_t)x * N * N_pad;
    double* W = Wall + (size_t)x * N * N_pad;
    for (int K = warp; K < R; K += 16) {
        const int c = order[(size_t)x * N + K];
        const double s = nrm[c], inv = s > 0 ? 1.0 / s : 0.0;
        for (int e = lane; e < N_pad; e += 32) {
            U[(size_t)K * N_pad + e] = (e < N) ? G[(size_t)c * N_pad + e] * inv : 0.0;
            W[(size_t)K * N_pad + e] = (e < N) ? V[(size_t)c * N_pad + e] : 0.0;
        }
    }
}

// ---- randomised range-finder SVD (LO_SETUP_RANDOMIZED_SVD), see gpu_pair_rsvd below.
// Gaussian test matrix Om[p][kk], p < N, kk < k, from the counter-based generator of lo_internal.h.
__global__ void k_gauss(double* __restrict__ Om, int N, int k, unsigned long long seed) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < N * k) Om[e] = gauss_at(seed, (unsigned long long)e);
}

// Small strided batched GEMM (setup only): C_x[i][j] = sum_l A_x(i,l) B_x(l,j), A_x(i,l) = A[x*a_b + i*a_i + l*a_l], same for
// B; 32 x 32 tile per CTA, 256 threads x 4 outputs.  resid != NULL: nothing is stored; instead the tile's
// sum_ij (D_x[i][j] - C_x[i][j])^2 goes to resid[(x * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x]  (D: ldc, batch d_b).
__global__ void __launch_bounds__(256) k_gemm_small(int M, int Nn, int K, const double* __restrict__ A, size_t a_b, int a_i, int a_l,
                                                    const double* __restrict__ B, size_t b_b, int b_l, int b_j, double* __restrict__ C,
                                                    size_t c_b, int ldc, const double* __restrict__ D, size_t d_b, double* __restrict__ resid) {
    __shared__ double As[32][33], Bs[32][33];
    __shared__ double red[8];
    const int x = blockIdx.z, i0 = blockIdx.y * 32, j0 = blockIdx.x * 32, tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double* Ax = A + x * a_b;
    const double* Bx = B + x * b_b;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int l0 = 0; l0 < K; l0 += 32) {
        __syncthreads();
        for (int e = threadIdx.x; e < 1024; e += 256) {
            const int r = e >> 5, c = e & 31;
            // As[r][c] = A(i0 + r, l0 + c): read along whichever index is contiguous
            const int ia = a_l == 1 ? r : c, la = a_l == 1 ? c : r;
            As[ia][la] = (i0 + ia < M && l0 + la < K) ? Ax[(size_t)(i0 + ia) * a_i + (size_t)(l0 + la) * a_l] : 0.0;
            const int lb = b_j == 1 ? r : c, jb = b_j == 1 ? c : r;
            Bs[lb][jb] = (l0 + lb < K && j0 + jb < Nn) ? Bx[(size_t)(l0 + lb) * b_l + (size_t)(j0 + jb) * b_j] : 0.0;
        }
        __syncthreads();
#pragma unroll 8
        for (int l = 0; l < 32; ++l) {
            const double b = Bs[l][tx];
#pragma unroll
            for (int u = 0; u < 4; ++u) acc[u] = fma(As[ty * 4 + u][l], b, acc[u]);
        }
    }
    if (!resid) {
        double* Cx = C + x * c_b;
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i0 + ty * 4 + u < M && j0 + tx < Nn) Cx[(size_t)(i0 + ty * 4 + u) * ldc + j0 + tx] = acc[u];
        return;
    }
    const double* Dx = D + x * d_b;
    double r2 = 0;
#pragma unroll
    for (int u = 0; u < 4; ++u)
        if (i0 + ty * 4 + u < M && j0 + tx < Nn) {
            const double d = Dx[(size_t)(i0 + ty * 4 + u) * ldc + j0 + tx] - acc[u];
            r2 = fma(d, d, r2);
        }
    r2 = warp_sum(r2);
    if (tx == 0) red[ty] = r2;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int q = 0; q < 8; ++q) t += red[q];
        resid[((size_t)x * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = t;
    }
}

// Rows of the orthogonalised sketch -> orthonormal basis rows: row / |row|, or 0 for a numerically null row (the sketch
// was wider than the block's rank; null relative to the longest row of the matrix).  Two passes, grid (k, n_mat), block 128.
__global__ void __launch_bounds__(128) k_row_len2(const double* __restrict__ Z, size_t stride, int k, int N, int N_pad, double* __restrict__ len2) {
    __shared__ double s_red[4];
    const double* row = Z + (size_t)blockIdx.y * stride + (size_t)blockIdx.x * N_pad;
    double a = 0;
    for (int e = threadIdx.x; e < N; e += 128) a = fma(row[e], row[e], a);
    a = warp_sum(a);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) len2[(size_t)blockIdx.y * k + blockIdx.x] = (s_red[0] + s_red[1]) + (s_red[2] + s_red[3]);
}
__global__ void __launch_bounds__(128) k_rows_scale(double* __restrict__ Z, size_t stride, int k, int N, int N_pad, const double* __restrict__ len2) {
    const double* l2 = len2 + (size_t)blockIdx.y * k;
    double longest = 0;
    for (int r = 0; r < k; ++r) longest = fmax(longest, l2[r]);
    const double tau = (double)N * 1.1102230246251565e-16, mine = l2[blockIdx.x];
    const double inv = mine > tau * tau * longest ? 1.0 / sqrt(mine) : 0.0;
    double* row = Z + (size_t)blockIdx.y * stride + (size_t)blockIdx.x * N_pad;
    for (int e = threadIdx.x; e < N_pad; e += 128) row[e] = (e < N) ? row[e] * inv : 0.0;
}

// packing: copy row blocks (whole rows of N_pad doubles, 16-byte vectors) according to a table
__global__ void __launch_bounds__(256) k_gather_rows(const double2* __restrict__ src, double2* __restrict__ dst, const GatherRec* __restrict__ table,
                                                     int half_pad) {
    const GatherRec rec = table[blockIdx.x];
    const double2* s = src + (size_t)rec.src_row * half_pad;
    double2* d = dst + (size_t)rec.dst_row * half_pad;
    const size_t n = (size_t)rec.r * half_pad;
    for (size_t e = threadIdx.x; e < n; e += 256) d[e] = s[e];
}

}  // namespace

lo_status gpu_gather_rows(const double* src, double* dst, const GatherRec* table, int n, int N_pad) {
    if (n <= 0) return LO_OK;
    GatherRec* d = nullptr;
    cudaError_t e = cudaMalloc(&d, (size_t)n * sizeof(GatherRec));
    if (e == cudaSuccess) e = cudaMemcpy(d, table, (size_t)n * sizeof(GatherRec), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_gather_rows<<<n, 256>>>(reinterpret_cast<const double2*>(src), reinterpret_cast<double2*>(dst), d, N_pad / 2);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (d) cudaFree(d);
    if (e != cudaSuccess) { set_error(std::string("gpu_gather_rows: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

// Randomised SVD of a batch of pair blocks (LO_SETUP_RANDOMIZED_SVD; "approximate versions of the singular value
// decomposition"), every step on the device; G = Y^T as left by k_pair_gram (rows = columns of Y):
//     Zt = Om^T G^T (k x N)            sketch of the column space of G with the Gaussian test matrix Om (N x k)
//     Pt = orth. rows of Zt            block Jacobi on the k rows, rows normalised (null rows -> 0)
//     Bp = Pt G  (k x N)               the block in that basis: G ~= Pt^T Bp
//     Vr Bp = diag(sigma) U            block Jacobi on the k rows of Bp, Vr accumulated  =>  Y ~= U^T diag(sigma) (Vr Pt)
//     resid = |G - (Vr Pt)^T (Vr Bp)|_F   formed explicitly: by Weyl every singular value of Y is within resid of a returned one
// A block is ACCEPTED when resid <= 16 N u |Y|_F (its numerical rank is below k, the result is the SVD to working
// accuracy); every other block of the batch is then decomposed by the full method in place.  The sketches live in the
// batch's V scratch (needs 4 k <= N).  accepted[x] tells the caller; counts go to stat.
lo_status gpu_pair_rsvd(const lo_factors* f, int spin, const int* pi, const int* pj, int n, int k, double* tmpY, double* tmpV, double* tmpU,
                        double* tmpW, double* dSigma, int* dOrder, double* hSigma, double skip_below, SvdStat* stat, long long* n_accepted) {
    const int N = f->N, N_pad = f->N_pad;
    const size_t mat = (size_t)N * N_pad;
    int *dpi = nullptr, *dpj = nullptr, *dSchedK = nullptr, *dSchedN = nullptr, *dSweeps = nullptr, *dIdx = nullptr;
    double *dOff = nullptr, *dOm = nullptr, *dLen2 = nullptr, *dRes = nullptr;
    const std::vector<int> schedK = svd_schedule((k + SVD_B - 1) / SVD_B), schedN = svd_schedule((N + SVD_B - 1) / SVD_B);
    const int tiles = (N + 31) / 32;
    std::vector<int> hSweeps(n), rej;
    std::vector<double> hOff(n), hRes((size_t)n * tiles * tiles);
    cudaError_t e = cudaSuccess;
    const char* where = "";
    auto step = [&](cudaError_t r, const char* w) { if (e == cudaSuccess && r != cudaSuccess) { e = r; where = w; } return e == cudaSuccess; };
    step(cudaMalloc(&dpi, (size_t)n * 4), "cudaMalloc") && step(cudaMalloc(&dpj, (size_t)n * 4), "cudaMalloc") &&
        step(cudaMalloc(&dSchedK, schedK.size() * 4), "cudaMalloc") && step(cudaMalloc(&dSchedN, schedN.size() * 4), "cudaMalloc") &&
        step(cudaMalloc(&dSweeps, (size_t)n * 4), "cudaMalloc") && step(cudaMalloc(&dIdx, (size_t)n * 4), "cudaMalloc") &&
        step(cudaMalloc(&dOff, (size_t)n * 8), "cudaMalloc") && step(cudaMalloc(&dOm, (size_t)N * k * 8), "cudaMalloc") &&
        step(cudaMalloc(&dLen2, (size_t)n * k * 8), "cudaMalloc") && step(cudaMalloc(&dRes, hRes.size() * 8), "cudaMalloc") &&
        step(cudaMemcpy(dpi, pi, (size_t)n * 4, cudaMemcpyHostToDevice), "cudaMemcpy") &&
        step(cudaMemcpy(dpj, pj, (size_t)n * 4, cudaMemcpyHostToDevice), "cudaMemcpy") &&
        step(cudaMemcpy(dSchedK, schedK.data(), schedK.size() * 4, cudaMemcpyHostToDevice), "cudaMemcpy") &&
        step(cudaMemcpy(dSchedN, schedN.data(), schedN.size() * 4, cudaMemcpyHostToDevice), "cudaMemcpy") &&
        step(cudaMemset(tmpV, 0, (size_t)n * mat * 8), "cudaMemset");
    double* Zt = tmpV;                                   // per pair x at x * mat: Zt/Pt [k][N_pad], Bp, Wf, Vr [k][k]
    double* Bp = tmpV + (size_t)k * N_pad;
    double* Wf = tmpV + (size_t)2 * k * N_pad;
    double* Vr = tmpV + (size_t)3 * k * N_pad;
    if (e == cudaSuccess) {
        dim3 grid((N_pad + 63) / 64, (N + 63) / 64, n);
        k_pair_gram<<<grid, 256>>>(f->ops->dLbar, f->n_chol, f->O_tot, N, N_pad, f->o_base[spin], dpi, dpj, tmpY);
        k_gauss<<<(N * k + 255) / 256, 256>>>(dOm, N, k, 0x2202008320000000ull + (unsigned long long)k);
        dim3 gk((N + 31) / 32, (k + 31) / 32, n), gn(tiles, tiles, n), gr(k, n);
        // Zt[kk][q] = sum_p Om[p][kk] G[q][p]
        k_gemm_small<<<gk, 256>>>(k, N, N, dOm, 0, 1, k, tmpY, mat, 1, N_pad, Zt, mat, N_pad, nullptr, 0, nullptr);
        step(cudaGetLastError(), "sketch");
        step(launch_block_jacobi(Zt, nullptr, n, k, N, N_pad, 0, dSchedK, -1.0, dSweeps, dOff, nullptr, mat, nullptr), "k_block_jacobi(sketch)");
        k_row_len2<<<gr, 128>>>(Zt, mat, k, N, N_pad, dLen2);
        k_rows_scale<<<gr, 128>>>(Zt, mat, k, N, N_pad, dLen2);
        // Bp[kk][c] = sum_q Pt[kk][q] G[q][c]
        k_gemm_small<<<gk, 256>>>(k, N, N, Zt, mat, N_pad, 1, tmpY, mat, N_pad, 1, Bp, mat, N_pad, nullptr, 0, nullptr);
        step(cudaGetLastError(), "project");
        step(launch_block_jacobi(Bp, Vr, n, k, N, N_pad, k, dSchedK, -1.0, dSweeps, dOff, nullptr, mat, nullptr), "k_block_jacobi(projected)");
        // Wf[K][q] = sum_kk Vr[K][kk] Pt[kk][q]
        k_gemm_small<<<gk, 256>>>(k, N, k, Vr, mat, k, 1, Zt, mat, N_pad, 1, Wf, mat, N_pad, nullptr, 0, nullptr);
        // resid^2 tiles of G - Wf^T Bp
        k_gemm_small<<<gn, 256>>>(N, N, k, Wf, mat, 1, N_pad, Bp, mat, N_pad, 1, nullptr, 0, N_pad, tmpY, mat, dRes);
        k_svd_finish<<<n, 512, (size_t)k * 8>>>(Bp, Wf, mat, k, N, N_pad, nullptr, dSigma, dOrder, tmpU, tmpW);
        step(cudaGetLastError(), "rsvd kernels");
    }
    step(cudaMemcpy(hSigma, dSigma, (size_t)n * N * 8, cudaMemcpyDeviceToHost), "cudaMemcpy(sigma)") &&
        step(cudaMemcpy(hSweeps.data(), dSweeps, (size_t)n * 4, cudaMemcpyDeviceToHost), "cudaMemcpy") &&
        step(cudaMemcpy(hOff.data(), dOff, (size_t)n * 8, cudaMemcpyDeviceToHost), "cudaMemcpy") &&
        step(cudaMemcpy(hRes.data(), dRes, hRes.size() * 8, cudaMemcpyDeviceToHost), "cudaMemcpy");
    if (e == cudaSuccess) {
        for (int x = 0; x < n; ++x) {
            double r2 = 0, s2 = 0;
            for (int t = 0; t < tiles * tiles; ++t) r2 += hRes[(size_t)x * tiles * tiles + t];
            for (int K = 0; K < k; ++K) s2 += hSigma[(size_t)x * N + K] * hSigma[(size_t)x * N + K];
            const bool ok = hSweeps[x] < SVD_MAX_SWEEPS && std::sqrt(r2) <= 16.0 * N * 1.1102230246251565e-16 * std::sqrt(s2 + r2);
            if (ok) { ++*n_accepted; stat->sweeps = std::max(stat->sweeps, hSweeps[x]); stat->offdiag = std::max(stat->offdiag, hOff[x]); }
            else rej.push_back(x);
        }
        if (!rej.empty()) {      // the blocks the sketch could not capture: the full method, in their own slots
            const int m = (int)rej.size();
            step(cudaMemcpy(dIdx, rej.data(), (size_t)m * 4, cudaMemcpyHostToDevice), "cudaMemcpy");
            step(launch_block_jacobi(tmpY, tmpV, m, N, N, N_pad, N_pad, dSchedN, skip_below, dSweeps, dOff, dIdx, mat, nullptr), "k_block_jacobi(full)");
            if (e == cudaSuccess) {
                k_svd_finish<<<m, 512, (size_t)N * 8>>>(tmpY, tmpV, mat, N, N, N_pad, dIdx, dSigma, dOrder, tmpU, tmpW);
                step(cudaGetLastError(), "k_svd_finish");
            }
            step(cudaMemcpy(hSigma, dSigma, (size_t)n * N * 8, cudaMemcpyDeviceToHost), "cudaMemcpy(sigma)") &&
                step(cudaMemcpy(hSweeps.data(), dSweeps, (size_t)n * 4, cudaMemcpyDeviceToHost), "cudaMemcpy") &&
                step(cudaMemcpy(hOff.data(), dOff, (size_t)n * 8, cudaMemcpyDeviceToHost), "cudaMemcpy");
            if (e == cudaSuccess)
                for (int x : rej) {
                    if (hSweeps[x] < 0) {
                        std::fill(hSigma + (size_t)x * N, hSigma + (size_t)(x + 1) * N, 0.0);
                        hSigma[(size_t)x * N] = hOff[x];
                        ++stat->screened;
                        continue;
                    }
                    stat->sweeps = std::max(stat->sweeps, hSweeps[x]);
                    stat->offdiag = std::max(stat->offdiag, hOff[x]);
                    if (hSweeps[x] >= SVD_MAX_SWEEPS) stat->converged = false;
                }
        }
    }
    cudaFree(dpi); cudaFree(dpj); cudaFree(dSchedK); cudaFree(dSchedN); cudaFree(dSweeps); cudaFree(dIdx); cudaFree(dOff); cudaFree(dOm);
    cudaFree(dLen2); cudaFree(dRes);
    if (e != cudaSuccess) { set_error(std::string("gpu_pair_rsvd: ") + where + ": " + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

size_t gpu_pair_svd_bytes_per_pair(int N, int N_pad) { return (size_t)4 * N * N_pad * 8 + (size_t)N * 12 + 16; }

lo_status gpu_pair_svd(const lo_factors* f, int spin, const int* pi, const int* pj, int n, double* tmpY, double* tmpV, double* tmpU,
                       double* tmpW, double* dSigma, int* dOrder, double* hSigma, double skip_below, SvdStat* stat) {
    const int N = f->N, N_pad = f->N_pad;
    int *dpi = nullptr, *dpj = nullptr, *dSched = nullptr, *dSweeps = nullptr;
    double* dOff = nullptr;
    const std::vector<int> sched = svd_schedule((N + SVD_B - 1) / SVD_B);
    std::vector<int> hSweeps(n);
    std::vector<double> hOff(n);
    cudaError_t e = cudaSuccess;
    const char* where = "";
    auto step = [&](cudaError_t r, const char* w) { if (e == cudaSuccess && r != cudaSuccess) { e = r; where = w; } return e == cudaSuccess; };
    step(cudaMalloc(&dpi, (size_t)n * 4), "cudaMalloc") && step(cudaMalloc(&dpj, (size_t)n * 4), "cudaMalloc") &&
        step(cudaMalloc(&dSched, sched.size() * 4), "cudaMalloc") && step(cudaMalloc(&dSweeps, (size_t)n * 4), "cudaMalloc") &&
        step(cudaMalloc(&dOff, (size_t)n * 8), "cudaMalloc") &&
        step(cudaMemcpy(dpi, pi, (size_t)n * 4, cudaMemcpyHostToDevice), "cudaMemcpy") &&
        step(cudaMemcpy(dpj, pj, (size_t)n * 4, cudaMemcpyHostToDevice), "cudaMemcpy") &&
        step(cudaMemcpy(dSched, sched.data(), sched.size() * 4, cudaMemcpyHostToDevice), "cudaMemcpy");
    if (e == cudaSuccess) {
        dim3 grid((N_pad + 63) / 64, (N + 63) / 64, n);
        k_pair_gram<<<grid, 256>>>(f->ops->dLbar, f->n_chol, f->O_tot, N, N_pad, f->o_base[spin], dpi, dpj, tmpY);
        step(cudaGetLastError(), "k_pair_gram");
    }
    if (e == cudaSuccess) step(launch_block_jacobi(tmpY, tmpV, n, N, N, N_pad, N_pad, dSched, skip_below, dSweeps, dOff, nullptr, (size_t)N * N_pad, nullptr), "k_block_jacobi");
    if (e == cudaSuccess) {
        k_svd_finish<<<n, 512, (size_t)N * 8>>>(tmpY, tmpV, (size_t)N * N_pad, N, N, N_pad, nullptr, dSigma, dOrder, tmpU, tmpW);
        step(cudaGetLastError(), "k_svd_finish");
    }
    step(cudaMemcpy(hSigma, dSigma, (size_t)n * N * 8, cudaMemcpyDeviceToHost), "cudaMemcpy(sigma)") &&
        step(cudaMemcpy(hSweeps.data(), dSweeps, (size_t)n * 4, cudaMemcpyDeviceToHost), "cudaMemcpy") &&
        step(cudaMemcpy(hOff.data(), dOff, (size_t)n * 8, cudaMemcpyDeviceToHost), "cudaMemcpy");
    cudaFree(dpi); cudaFree(dpj); cudaFree(dSched); cudaFree(dSweeps); cudaFree(dOff);      // on every path
    if (e != cudaSuccess) { set_error(std::string("gpu_pair_svd: ") + where + ": " + cudaGetErrorString(e)); return LO_ECUDA; }
    for (int x = 0; x < n; ++x) {
        if (hSweeps[x] < 0) {           // screened by |Y|_F <= threshold: sigma_1 reported as that bound, everything else 0
            std::fill(hSigma + (size_t)x * N, hSigma + (size_t)(x + 1) * N, 0.0);
            hSigma[(size_t)x * N] = hOff[x];
            ++stat->screened;
            continue;
        }
        stat->sweeps = std::max(stat->sweeps, hSweeps[x]);
        stat->offdiag = std::max(stat->offdiag, hOff[x]);
        if (hSweeps[x] >= SVD_MAX_SWEEPS) stat->converged = false;
    }
    return LO_OK;
}

}  // namespace lo
