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

// sigma_K = |g_{order[K]}| descending;  U row K = g/sigma;  W row K = v.
__global__ void __launch_bounds__(512) k_svd_finish(const double* __restrict__ Gall, const double* __restrict__ Vall, int N, int N_pad,
                                                    double* __restrict__ sigma, int* __restrict__ order, double* __restrict__ Uall,
                                                    double* __restrict__ Wall) {
    extern __shared__ double nrm[];   // [N]
    const int x = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* G = Gall + (size_t)x * N * N_pad;
    const double* V = Vall + (size_t)x * N * N_pad;
    for (int c = warp; c < N; c += 16) {
        double a = 0;
        for (int e = lane; e < N; e += 32) { double g = G[(size_t)c * N_pad + e]; a = fma(g, g, a); }
        a = warp_sum(a);
        if (lane == 0) nrm[c] = sqrt(a);
    }
    __syncthreads();
    for (int c = tid; c < N; c += 512) {
        const double v = nrm[c];
        int rank = 0;
        for (int d = 0; d < N; ++d) {
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
    for (int K = warp; K < N; K += 16) {
        const int c = order[(size_t)x * N + K];
        const double s = nrm[c], inv = s > 0 ? 1.0 / s : 0.0;
        for (int e = lane; e < N_pad; e += 32) {
            U[(size_t)K * N_pad + e] = (e < N) ? G[(size_t)c * N_pad + e] * inv : 0.0;
            W[(size_t)K * N_pad + e] = (e < N) ? V[(size_t)c * N_pad + e] : 0.0;
        }
    }
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
    if (e == cudaSuccess) step(launch_block_jacobi(tmpY, tmpV, n, N, N_pad, dSched, skip_below, dSweeps, dOff, nullptr), "k_block_jacobi");
    if (e == cudaSuccess) {
        k_svd_finish<<<n, 512, (size_t)N * 8>>>(tmpY, tmpV, N, N_pad, dSigma, dOrder, tmpU, tmpW);
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
