// lo_setup_gpu.cu -- device side of lo_setup (flag LO_SETUP_GPU_SVD): pair blocks Y^{ij} and their
// SVDs (Eq. 18) by a batched one-sided (Hestenes) Jacobi method, one CTA per pair block.
// Setup is untimed; these kernels are written for robustness and a bounded run time at the
// pentacene-sized config (2701 SVDs of 378 x 378), not for roofline.
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

// One CTA (512 threads = 16 warps) per matrix.  Vectors g_c = G[c][0..N) are orthogonalised by plane rotations in
// round-robin (tournament) order, N/2 disjoint pairs per round spread over the warps; V accumulates the rotations.
__global__ void __launch_bounds__(512) k_jacobi(double* __restrict__ Gall, double* __restrict__ Vall, int N, int N_pad, int max_sweeps,
                                                int* __restrict__ sweeps_out) {
    __shared__ int s_rot;
    __shared__ double s_red[16];
    __shared__ double s_tiny2;
    const int x = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* G = Gall + (size_t)x * N * N_pad;
    double* V = Vall + (size_t)x * N * N_pad;
    // V = I, Frobenius norm
    double fro = 0;
    for (size_t e = tid; e < (size_t)N * N_pad; e += 512) {
        int r = (int)(e / N_pad), c = (int)(e % N_pad);
        V[e] = (r == c) ? 1.0 : 0.0;
        double g = G[e];
        fro += g * g;
    }
    fro = warp_sum(fro);
    if (lane == 0) s_red[warp] = fro;
    __syncthreads();
    if (tid == 0) {
        double t = 0;
        for (int q = 0; q < 16; ++q) t += s_red[q];
        s_tiny2 = t * 1e-30;
    }
    __syncthreads();
    const double tiny2 = s_tiny2, tol = 1e-15;
    const int m = N + (N & 1);
    int sweep = 0;
    for (; sweep < max_sweeps; ++sweep) {
        if (tid == 0) s_rot = 0;
        __syncthreads();
        int myrot = 0;
        for (int round = 0; round < m - 1; ++round) {
            for (int k = warp; k < m / 2; k += 16) {
                int p, q;
                if (k == 0) { p = m - 1; q = round; }
                else { p = (round + k) % (m - 1); q = (round - k + (m - 1)) % (m - 1); }
                if (p >= N || q >= N) continue;
                if (p > q) { int t = p; p = q; q = t; }
                double* gp = G + (size_t)p * N_pad;
                double* gq = G + (size_t)q * N_pad;
                double a = 0, b = 0, c = 0;
                for (int e = lane; e < N; e += 32) {
                    double xx = gp[e], yy = gq[e];
                    a = fma(xx, xx, a); b = fma(yy, yy, b); c = fma(xx, yy, c);
                }
                a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
                if (a <= tiny2 || b <= tiny2) continue;
                if (fabs(c) <= tol * sqrt(a * b)) continue;
                ++myrot;
                const double zeta = (b - a) / (2.0 * c);
                const double t = (zeta >= 0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
                double* vp = V + (size_t)p * N_pad;
                double* vq = V + (size_t)q * N_pad;
                for (int e = lane; e < N; e += 32) {
                    double xx = gp[e], yy = gq[e];
                    gp[e] = cs * xx - sn * yy;
                    gq[e] = sn * xx + cs * yy;
                    double vx = vp[e], vy = vq[e];
                    vp[e] = cs * vx - sn * vy;
                    vq[e] = sn * vx + cs * vy;
                }
            }
            __syncthreads();
        }
        if (lane == 0 && myrot) atomicAdd(&s_rot, myrot);
        __syncthreads();
        const int rot = s_rot;
        __syncthreads();
        if (rot == 0) break;
    }
    if (tid == 0 && sweeps_out) sweeps_out[x] = sweep;
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

size_t gpu_pair_svd_bytes_per_pair(int N, int N_pad) { return (size_t)4 * N * N_pad * 8 + (size_t)N * 12; }

lo_status gpu_pair_svd(const lo_factors* f, int spin, const int* pi, const int* pj, int n, double* tmpY, double* tmpV, double* tmpU,
                       double* tmpW, double* dSigma, int* dOrder, double* hSigma) {
#define GK(call)                                                                                      \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess) { set_error(std::string(#call) + ": " + cudaGetErrorString(e_)); return LO_ECUDA; } \
    } while (0)
    const int N = f->N, N_pad = f->N_pad;
    int *dpi = nullptr, *dpj = nullptr;
    GK(cudaMalloc(&dpi, (size_t)n * 4));
    GK(cudaMalloc(&dpj, (size_t)n * 4));
    GK(cudaMemcpy(dpi, pi, (size_t)n * 4, cudaMemcpyHostToDevice));
    GK(cudaMemcpy(dpj, pj, (size_t)n * 4, cudaMemcpyHostToDevice));
    dim3 grid((N_pad + 63) / 64, (N + 63) / 64, n);
    k_pair_gram<<<grid, 256>>>(f->ops->dLbar, f->n_chol, f->O_tot, N, N_pad, f->o_base[spin], dpi, dpj, tmpY);
    GK(cudaGetLastError());
    k_jacobi<<<n, 512>>>(tmpY, tmpV, N, N_pad, 60, nullptr);
    GK(cudaGetLastError());
    k_svd_finish<<<n, 512, (size_t)N * 8>>>(tmpY, tmpV, N, N_pad, dSigma, dOrder, tmpU, tmpW);
    GK(cudaGetLastError());
    GK(cudaMemcpy(hSigma, dSigma, (size_t)n * N * 8, cudaMemcpyDeviceToHost));
    cudaFree(dpi);
    cudaFree(dpj);
    return LO_OK;
#undef GK
}

}  // namespace lo
