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
//   k_cas_*     multi-determinant trial (NEXT-2): SMW overlaps / Green's functions (k_cas_T, k_cas_coef, k_cas_theta),
//               rearranged SMW energy (k_cas_pairs, k_cas_H, k_cas_energy, k_cas_e1sum), k_cas_combine
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

namespace lo {

namespace {

__device__ __forceinline__ void mma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// Stage release must not overtake the stage's shared-memory reads.  ptxas is free to sink register-only MMAs below the
// mbarrier arrive, and then the last ld.shared of a stage can still be in flight when the arrive issues (the arrive goes
// through the SYNCS unit, not the load pipe) and the producer's TMA refill (async proxy) can land first -- seen as rare
// wrong rows of X at configs[3].  release_stage() is the documented ordering for generic-proxy reads followed by an
// async-proxy overwrite: fence.proxy.async (SASS: MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC, waits for the warp's outstanding
// loads), then the arrive.  It is issued right after the LAST fragment loads of a stage and before their MMAs, so the
// wait overlaps the MMAs still queued on the tensor pipe.
// ---- TMA + mbarrier plumbing (cp.async.bulk.tensor; SASS: UTMALDG / SYNCS)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void release_stage(uint32_t empty_bar, int lane) {
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(empty_bar);
}
// Warp-specialised register budget (setmaxnreg, per warpgroup): the kernels launch 3 warpgroups at 168 registers per
// thread; the producer warpgroup shrinks to 40, the two consumer warpgroups grow to 232 (4*32*40 + 8*32*232 = 64512).
__device__ __forceinline__ void reg_dec_producer() { asm volatile("setmaxnreg.dec.sync.aligned.u32 40;"); }
__device__ __forceinline__ void reg_inc_consumer() { asm volatile("setmaxnreg.inc.sync.aligned.u32 232;"); }
__device__ __forceinline__ void bar_sync_consumers() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// 2D tiled TMA load: box [rows][16 doubles] at (k0 = inner coordinate in doubles, row0) -> 128-byte-swizzled smem tile
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int k0, int row0, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(k0), "r"(row0), "r"(bar) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* tm) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tm)) : "memory");
}
// Ampere-style asynchronous copies (LDGSTS) for the S1 staging; src_size 0 zero-fills the destination
__device__ __forceinline__ void cp_async8(void* dst, const void* src, bool valid) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(valid ? 8 : 0) : "memory");
}
__device__ __forceinline__ void cp_async16(void* dst, const void* src, bool valid) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(dst)), "l"(src), "r"(valid ? 16 : 0) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }
__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// Shared-memory operand tiles are [rows][16 doubles] = 128 bytes per row, written by TMA with the 128-byte swizzle:
// the 16-byte chunk c of row r lands at chunk c ^ (r & 7) (tile base 1024-byte aligned).  MMA k-step s (0..3) of a
// K tile takes the logical k indices {2s, 2s+1, 2s+8, 2s+9} for t = 0..3 -- the same permutation for A and B, so the
// contraction is unchanged -- which puts the 16 lanes of a half-warp (4 rows x 4 k) on 16 distinct 8-byte banks.
// frag_off(g, t, s): byte offset inside a row whose (r & 7) == g.
__device__ __forceinline__ uint32_t frag_off(int g, int t, int s) {
    return (uint32_t)((((s + 4 * (t >> 1)) ^ g) << 4) + (t & 1) * 8);
}

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
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 crecip(double2 a) {
    // Smith's algorithm with correctly rounded reciprocals (MUFU.RCP64H + Newton) instead of the two divisions: the
    // reciprocal sits on the serial chain of every Gauss-Jordan step
    if (fabs(a.x) >= fabs(a.y)) {
        const double r = a.y * __drcp_rn(a.x), id = __drcp_rn(a.x + a.y * r);
        return make_double2(id, -r * id);
    } else {
        const double r = a.x * __drcp_rn(a.y), id = __drcp_rn(a.x * r + a.y);
        return make_double2(r * id, -id);
    }
}

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
template <bool RAGGED>
__global__ void __launch_bounds__(384, 1) k_coulomb(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmT,
                                                    double* __restrict__ Xpart, int Xp, int O_tot, int N_pad, int ldw, int RB, int NB,
                                                    int nsplit, int n_cols) {
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
                    mbar_expect_tx(bar, CO_STAGE_BYTES);
                    tma_load_2d(st, &tmA, o * N_pad + kt * KTILE, it.rb * CO_BM, bar);
                    tma_load_2d(st + CO_BM * 128, &tmT, kt * KTILE, o * ldw + it.nb * 128, bar);
                    if (++slot == CO_STAGES) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }
    // ===== 8 consumer warps (64 x 32 each)
    reg_inc_consumer();
    const int cw = warp - 4, g = lane >> 2, t = lane & 3, wm = RAGGED ? (cw & 1) : (cw >> 2), wn = RAGGED ? (cw >> 1) : (cw & 3);
    double acc[8][4][2];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t a_row = (uint32_t)(wm * 64 + g) * 128, b_row = (uint32_t)(CO_BM + wn * 32 + g) * 128;
    int cslot = 0;
    uint32_t cphase = 0;
    for (long long q = blockIdx.x; q < n_items; q += gridDim.x) {
        const CoItem it = co_item(q, RB, NB, nsplit, ksteps);
        if (RAGGED && it.nb * 128 + wn * 32 >= n_cols) {          // warp-uniform: no walker in this warp's 32 columns
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
                double a[8], b[4];
#pragma unroll
                for (int mf = 0; mf < 8; ++mf) a[mf] = lds_f64(st + a_row + mf * 1024 + xo[ks]);
#pragma unroll
                for (int nf = 0; nf < 4; ++nf) b[nf] = lds_f64(st + b_row + nf * 1024 + xo[ks]);
                if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                for (int mf = 0; mf < 8; ++mf)
#pragma unroll
                    for (int nf = 0; nf < 4; ++nf) mma884(acc[mf][nf][0], acc[mf][nf][1], a[mf], b[nf]);
            }
            if (++cslot == CO_STAGES) { cslot = 0; cphase ^= 1; }
        }
        double* Xs = Xpart + (size_t)it.sp * Xp * ldw;
#pragma unroll
        for (int mf = 0; mf < 8; ++mf)
#pragma unroll
            for (int nf = 0; nf < 4; ++nf) {
                int row = it.rb * CO_BM + wm * 64 + mf * 8 + g;
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
// small-rank workload).  4-stage TMA/mbarrier pipeline running across items; a short tile loads only its own 8-row
// fragments of U and W.  The C fragment holds (re, im) of one walker in one lane, for a and b alike, so the complex
// product is lane-local; rows are reduced by warp shuffles.  Persistent CTAs with a static round-robin schedule and
// per-CTA partial sums accumulated in a fixed order -> bitwise repeatable.
constexpr int EX_STAGES = 4;
constexpr int EX_STAGE_BYTES = (2 * EX_BM + 2 * 128) * 128;
constexpr int EX_RING = 8;      // tile-descriptor ring (producer -> consumers), > EX_STAGES items can never be in flight
constexpr int EX_SMEM = EX_STAGES * EX_STAGE_BYTES + 1024 + 128 + EX_RING * 16;

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
__global__ void __launch_bounds__(384, 1) k_exchange(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmW,
                                                     const __grid_constant__ CUtensorMap tmU8, const __grid_constant__ CUtensorMap tmW8,
                                                     const __grid_constant__ CUtensorMap tmT, const double* __restrict__ wgt,
                                                     const ExTile* __restrict__ tiles, long long n_items, int NB, int N_pad, int ldw,
                                                     double* __restrict__ ekpart, double* __restrict__ ejpart, int Wcap, int n_w) {
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
        prefetch_tmap(&tmU);
        prefetch_tmap(&tmW);
        prefetch_tmap(&tmU8);
        prefetch_tmap(&tmW8);
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
            for (long long q = blockIdx.x; q < n_items; q += gridDim.x, ++n) {
                const ExTile tile = tiles[q / NB];
                const int nb = (int)(q % NB);
                const uint32_t tx = (uint32_t)(2 * tile.nfrag * 8 + 2 * 128) * 128;
                for (int kt = 0; kt < KT; ++kt) {
                    mbar_wait(empty + 8 * slot, phase ^ 1);
                    if (kt == 0) ring[n % EX_RING] = tile;      // ordered before the consumers' wait by arrive.expect_tx (release)
                    const uint32_t st = sbase + slot * EX_STAGE_BYTES, bar = full + 8 * slot;
                    const int k0 = kt * KTILE;
                    mbar_expect_tx(bar, tx);
                    if (tile.nfrag == EX_BM / 8) {
                        tma_load_2d(st, &tmU, k0, tile.row0, bar);
                        tma_load_2d(st + EX_BM * 128, &tmW, k0, tile.row0, bar);
                    } else {
                        for (int fr = 0; fr < tile.nfrag; ++fr) {
                            tma_load_2d(st + fr * 1024, &tmU8, k0, tile.row0 + fr * 8, bar);
                            tma_load_2d(st + EX_BM * 128 + fr * 1024, &tmW8, k0, tile.row0 + fr * 8, bar);
                        }
                    }
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
    for (long long q = blockIdx.x; q < n_items; q += gridDim.x, ++n) {
        const int nb = (int)(q % NB);
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
// columns) and the warps split the ROW fragments instead: warp cw owns column half cw & 1 (8 walkers) and fragments
// cw >> 1 and 4 + (cw >> 1).  Same TMA/mbarrier pipeline (6 stages of 24 KB); the four fragment groups of a column half
// are added in a fixed order through shared memory.
constexpr int EN_STAGES = 6;
constexpr int EN_STAGE_BYTES = (2 * EX_BM + 2 * 32) * 128;
constexpr int EN_SMEM = EN_STAGES * EN_STAGE_BYTES + 1024 + 128 + EX_RING * 16 + 4 * 32 * 8;

__global__ void __launch_bounds__(384, 1) k_exchange_narrow(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmW,
                                                            const __grid_constant__ CUtensorMap tmU8, const __grid_constant__ CUtensorMap tmW8,
                                                            const __grid_constant__ CUtensorMap tmT32, const double* __restrict__ wgt,
                                                            const ExTile* __restrict__ tiles, long long n_items, int NB, int N_pad, int ldw,
                                                            double* __restrict__ ekpart, int Wcap) {
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const uint32_t full = sbase + EN_STAGES * EN_STAGE_BYTES, empty = full + 8 * EN_STAGES;
    ExTile* ring = reinterpret_cast<ExTile*>(sgen + EN_STAGES * EN_STAGE_BYTES + 128);
    double* red = reinterpret_cast<double*>(sgen + EN_STAGES * EN_STAGE_BYTES + 128 + EX_RING * 16);      // [4 fragment groups][32 columns]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KT = N_pad / KTILE;
    double* mypart = ekpart + (size_t)blockIdx.x * 2 * Wcap;
    for (int i = tid; i < 2 * Wcap; i += 384) mypart[i] = 0.0;
    if (tid == 0) {
        prefetch_tmap(&tmU);
        prefetch_tmap(&tmW);
        prefetch_tmap(&tmU8);
        prefetch_tmap(&tmW8);
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
            for (long long q = blockIdx.x; q < n_items; q += gridDim.x, ++n) {
                const ExTile tile = tiles[q / NB];
                const int nb = (int)(q % NB);
                // whole 64-row boxes of U and W whatever the tile's length (rows past the tile are never read): 4 TMA
                // issues per 24 KB stage -- a narrow item has too little MMA work per stage to hide more
                const uint32_t tx = (uint32_t)(2 * EX_BM + 2 * 32) * 128;
                for (int kt = 0; kt < KT; ++kt) {
                    mbar_wait(empty + 8 * slot, phase ^ 1);
                    if (kt == 0) ring[n % EX_RING] = tile;
                    const uint32_t st = sbase + slot * EN_STAGE_BYTES, bar = full + 8 * slot;
                    const int k0 = kt * KTILE;
                    mbar_expect_tx(bar, tx);
                    tma_load_2d(st, &tmU, k0, tile.row0, bar);
                    tma_load_2d(st + EX_BM * 128, &tmW, k0, tile.row0, bar);
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
    const int cg = cw & 1, fr0 = cw >> 1, fr1 = 4 + (cw >> 1);
    double accA[2][2][2], accB[2][2][2];
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int b = 0; b < 2; ++b) accA[j][b][0] = accA[j][b][1] = accB[j][b][0] = accB[j][b][1] = 0.0;
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t u_row0 = (uint32_t)(fr0 * 8 + g) * 128, u_row1 = (uint32_t)(fr1 * 8 + g) * 128;
    const uint32_t tj_row = (uint32_t)(2 * EX_BM + cg * 16 + g) * 128, ti_row = tj_row + 32 * 128;
    int cslot = 0, n = 0;
    uint32_t cphase = 0;
    for (long long q = blockIdx.x; q < n_items; q += gridDim.x, ++n) {
        const int nb = (int)(q % NB);
        mbar_wait(full + 8 * cslot, cphase);
        const ExTile tile = ring[n % EX_RING];
        const int nu = (fr0 < tile.nfrag ? 1 : 0) + (fr1 < tile.nfrag ? 1 : 0);     // warp-uniform
        for (int kt = 0; kt < KT; ++kt) {
            if (kt) mbar_wait(full + 8 * cslot, cphase);
            const uint32_t st = sbase + cslot * EN_STAGE_BYTES;
            if (nu > 0) {
#pragma unroll
                for (int ks = 0; ks < KTILE / 4; ++ks) {
                    double a[2], w[2], bj[2], bi[2];
                    a[0] = lds_f64(st + u_row0 + xo[ks]);
                    w[0] = lds_f64(st + u_row0 + EX_BM * 128 + xo[ks]);
                    if (nu == 2) {
                        a[1] = lds_f64(st + u_row1 + xo[ks]);
                        w[1] = lds_f64(st + u_row1 + EX_BM * 128 + xo[ks]);
                    }
#pragma unroll
                    for (int nf = 0; nf < 2; ++nf) {
                        bj[nf] = lds_f64(st + tj_row + nf * 1024 + xo[ks]);
                        bi[nf] = lds_f64(st + ti_row + nf * 1024 + xo[ks]);
                    }
                    if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                    for (int nf = 0; nf < 2; ++nf) {
                        mma884(accA[0][nf][0], accA[0][nf][1], a[0], bj[nf]);
                        mma884(accB[0][nf][0], accB[0][nf][1], w[0], bi[nf]);
                    }
                    if (nu == 2) {
#pragma unroll
                        for (int nf = 0; nf < 2; ++nf) {
                            mma884(accA[1][nf][0], accA[1][nf][1], a[1], bj[nf]);
                            mma884(accB[1][nf][0], accB[1][nf][1], w[1], bi[nf]);
                        }
                    }
                }
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + 8 * cslot);
            }
            if (++cslot == EN_STAGES) { cslot = 0; cphase ^= 1; }
        }
        double e[2][2];
#pragma unroll
        for (int nf = 0; nf < 2; ++nf) e[nf][0] = e[nf][1] = 0.0;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const double wv = j < nu ? __ldg(wgt + tile.row0 + (j == 0 ? fr0 : fr1) * 8 + g) : 0.0;
#pragma unroll
            for (int nf = 0; nf < 2; ++nf) {
                const double ar = accA[j][nf][0], ai = accA[j][nf][1], br = accB[j][nf][0], bi = accB[j][nf][1];
                e[nf][0] = fma(wv, ar * br - ai * bi, e[nf][0]);
                e[nf][1] = fma(wv, ar * bi + ai * br, e[nf][1]);
                accA[j][nf][0] = accA[j][nf][1] = accB[j][nf][0] = accB[j][nf][1] = 0.0;
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
                if (g == 0) red[(cw >> 1) * 32 + cg * 16 + nf * 8 + 2 * t + c] = v;
            }
        bar_sync_consumers();
        if (ctid < 32) mypart[(size_t)nb * 32 + ctid] += (red[ctid] + red[32 + ctid]) + (red[64 + ctid] + red[96 + ctid]);
        bar_sync_consumers();
    }
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
// and a determinant's pair energies are small bilinear forms in S (k_cas_energy).  Work item = (row tile, block of 8
// walkers); consumer warp m owns row fragment m and all NP panels x 16 real columns; same TMA/mbarrier pipeline.
constexpr int CP_STAGES = 4;
template <int NP>
struct CpCfg {
    static constexpr int STAGE_BYTES = 2 * EX_BM * 128 + NP * 16 * 128;
    static constexpr int SL = NP * NP + 1;      // slice stride (double2) of one (row group, walker): odd, so the 8 lanes of a
                                                // 128-bit shared access land on distinct 16-byte bank groups
    static constexpr int SMEM = CP_STAGES * STAGE_BYTES + 1024 + 128 + EX_RING * 16 + 8 * 8 * SL * 16;
};

template <int NP>
__global__ void __launch_bounds__(384, 1) k_cas_pairs(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmW,
                                                      const __grid_constant__ CUtensorMap tmT0, const double* __restrict__ wgt,
                                                      const ExTile* __restrict__ tiles, long long n_items, int WB, int N_pad, int ldw0,
                                                      const int* __restrict__ act /* [NP-2] */, double2* __restrict__ S, int n_w) {
    constexpr int STAGE = CpCfg<NP>::STAGE_BYTES;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    unsigned char* sgen = smem_raw + (sbase - smem_u32(smem_raw));
    const uint32_t full = sbase + CP_STAGES * STAGE, empty = full + 8 * CP_STAGES;
    ExTile* ring = reinterpret_cast<ExTile*>(sgen + CP_STAGES * STAGE + 128);
    double2* Sacc = reinterpret_cast<double2*>(sgen + CP_STAGES * STAGE + 128 + EX_RING * 16);     // [8 fragments (warps)][8 walkers][SL]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KT = N_pad / KTILE;
    if (tid == 0) {
        prefetch_tmap(&tmU);
        prefetch_tmap(&tmW);
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
            for (long long q = blockIdx.x; q < n_items; q += gridDim.x, ++n) {
                const ExTile tile = tiles[q / WB];
                const int wb = (int)(q % WB);
                pan[0] = tile.pi;
                pan[1] = tile.pj;
                // whole 64-row boxes of U and W whatever the tile's length (rows past the tile are never read): one TMA each
                const uint32_t tx = (uint32_t)(2 * EX_BM + NP * 16) * 128;
                for (int kt = 0; kt < KT; ++kt) {
                    mbar_wait(empty + 8 * slot, phase ^ 1);
                    if (kt == 0) ring[n % EX_RING] = tile;
                    const uint32_t st = sbase + slot * STAGE, bar = full + 8 * slot;
                    const int k0 = kt * KTILE;
                    mbar_expect_tx(bar, tx);
                    tma_load_2d(st, &tmU, k0, tile.row0, bar);
                    tma_load_2d(st + EX_BM * 128, &tmW, k0, tile.row0, bar);
#pragma unroll
                    for (int c = 0; c < NP; ++c)        // 16 real rows (8 walkers) of panel c
                        tma_load_2d(st + 2 * EX_BM * 128 + c * 2048, &tmT0, k0, pan[c] * ldw0 + wb * 16, bar);
                    if (++slot == CP_STAGES) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }
    reg_inc_consumer();
    // Work units of an item = (row fragment, column half nf) = 2 * nfrag; consumer warp cw owns units cw and cw + 8, i.e.
    // fragments cw/2 and 4 + cw/2 of the SAME column half nf = cw & 1 (they share the panel fragments).  The two warps
    // of a scheduler (cw, cw + 4) then hold at most ceil(nfrag / 2) + ... units: 5 fragments load the four schedulers
    // 3/3/2/2 instead of 2/1/1/1 whole fragments.
    const int cw = warp - 4, g = lane >> 2, t = lane & 3, ctid = tid - 128;
    const int nf = cw & 1, fr0 = cw >> 1, fr1 = 4 + (cw >> 1);
    double accU[2][NP][2], accW[2][NP][2];
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int c = 0; c < NP; ++c) accU[j][c][0] = accU[j][c][1] = accW[j][c][0] = accW[j][c][1] = 0.0;
    uint32_t xo[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) xo[s] = frag_off(g, t, s);
    const uint32_t u_row0 = (uint32_t)(fr0 * 8 + g) * 128, u_row1 = (uint32_t)(fr1 * 8 + g) * 128;
    const uint32_t p_row = (uint32_t)(2 * EX_BM * 128) + (uint32_t)(nf * 8 + g) * 128;
    constexpr int SL = CpCfg<NP>::SL;
    int cslot = 0, n = 0;
    uint32_t cphase = 0;
    for (long long q = blockIdx.x; q < n_items; q += gridDim.x, ++n) {
        const int wb = (int)(q % WB);
        const long long tix = q / WB;
        mbar_wait(full + 8 * cslot, cphase);
        const ExTile tile = ring[n % EX_RING];
        const int nu = (fr0 < tile.nfrag ? 1 : 0) + (fr1 < tile.nfrag ? 1 : 0);     // warp-uniform: 0, 1 or 2 units
        for (int kt = 0; kt < KT; ++kt) {
            if (kt) mbar_wait(full + 8 * cslot, cphase);
            const uint32_t st = sbase + cslot * STAGE;
            if (nu == 2) {
#pragma unroll
                for (int ks = 0; ks < KTILE / 4; ++ks) {
                    const double a0 = lds_f64(st + u_row0 + xo[ks]), w0 = lds_f64(st + u_row0 + EX_BM * 128 + xo[ks]);
                    const double a1 = lds_f64(st + u_row1 + xo[ks]), w1 = lds_f64(st + u_row1 + EX_BM * 128 + xo[ks]);
                    double bb[NP];
#pragma unroll
                    for (int c = 0; c < NP; ++c) bb[c] = lds_f64(st + p_row + c * 2048 + xo[ks]);
                    if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                    for (int c = 0; c < NP; ++c) {
                        mma884(accU[0][c][0], accU[0][c][1], a0, bb[c]);
                        mma884(accW[0][c][0], accW[0][c][1], w0, bb[c]);
                        mma884(accU[1][c][0], accU[1][c][1], a1, bb[c]);
                        mma884(accW[1][c][0], accW[1][c][1], w1, bb[c]);
                    }
                }
            } else if (nu == 1) {
#pragma unroll
                for (int ks = 0; ks < KTILE / 4; ++ks) {
                    const double a0 = lds_f64(st + u_row0 + xo[ks]), w0 = lds_f64(st + u_row0 + EX_BM * 128 + xo[ks]);
                    double bb[NP];
#pragma unroll
                    for (int c = 0; c < NP; ++c) bb[c] = lds_f64(st + p_row + c * 2048 + xo[ks]);
                    if (ks == KTILE / 4 - 1) release_stage(empty + 8 * cslot, lane);
#pragma unroll
                    for (int c = 0; c < NP; ++c) {
                        mma884(accU[0][c][0], accU[0][c][1], a0, bb[c]);
                        mma884(accW[0][c][0], accW[0][c][1], w0, bb[c]);
                    }
                }
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + 8 * cslot);
            }
            if (++cslot == CP_STAGES) { cslot = 0; cphase ^= 1; }
        }
        // epilogue: S[c][c'] of the 4 walkers of this warp's column half, per unit.  For every panel c the lane holds the 8
        // complex products of its own row g (c' = 0..7, zero beyond NP); a transposing butterfly over the 8 row groups
        // (each round sends half of the values and keeps the other half: 8+4+2 exchanges instead of 3 per value) leaves
        // the row sum of column c' = 4 b0 + 2 b1 + b2 (bits of g) in lane g.  Every fragment's S goes to its own slice;
        // the slices are added in fragment order when the block is written out (fixed order).
        {
            const bool b0 = g & 1, b1 = g & 2, b2 = g & 4;
            const int c2own = (b0 ? 4 : 0) + (b1 ? 2 : 0) + (b2 ? 1 : 0);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                if (j >= nu) break;                     // warp-uniform
                const int fr = j == 0 ? fr0 : fr1;
                const double wv = __ldg(wgt + tile.row0 + fr * 8 + g);
                double2* dst = Sacc + ((fr * 8) + nf * 4 + t) * SL;
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
                    if (c2own < NP) dst[c * NP + c2own] = make_double2(v[0], v[1]);
                }
#pragma unroll
                for (int c = 0; c < NP; ++c) accU[j][c][0] = accU[j][c][1] = accW[j][c][0] = accW[j][c][1] = 0.0;
            }
        }
        bar_sync_consumers();
        for (int i = ctid; i < 8 * NP * NP; i += 256) {
            const int wl = i / (NP * NP), wg = wb * 8 + wl;
            const int is = wl * SL + (i - wl * NP * NP);
            double2 sum = Sacc[is];
            for (int fr = 1; fr < tile.nfrag; ++fr) { const double2 v = Sacc[fr * 8 * SL + is]; sum.x += v.x; sum.y += v.y; }
            if (wg < n_w) S[((size_t)tix * n_w + wg) * NP * NP + (i - wl * NP * NP)] = sum;
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
        if (lane == 0) H[((size_t)w * n_orb + x) * 9 + sl] = make_double2(sr, si);
    }
}

// Pair energies of every determinant from the S intermediates (Eq. 22 with Eq. 23 inserted): with
// Theta^d_x = s_x Theta0_x + sum_k G_d[k][x] Theta0_{h_k}  (s_x = 1 for a reference non-hole, else 0),
//   exchange  e = sum_{c in y-list} sum_{c' in x-list} coef_y[c] coef_x[c'] S[c][c'],
//   Coulomb   j = sum_{c in x-list} sum_{c' in y-list} coef_x[c] coef_y[c'] S[c][c'],
// lists = {self, the determinant's holes}.  grid (n_chunks, n_w); a chunk of CE_CH tiles sits in shared memory, threads
// run over determinants; partial (E_K, E_J) sums per chunk are added in chunk order by k_cas_e1sum.
constexpr int CE_CH = 16;
template <int MAXE>     // compile-time bound of the excitation rank: the coefficient lists stay in registers
__global__ void __launch_bounds__(128) k_cas_energy(const double2* __restrict__ S, const ExTile* __restrict__ tiles, long long n_tiles,
                                                    const signed char* __restrict__ kind, const int* __restrict__ holeIdx,
                                                    const double2* __restrict__ G, double2* __restrict__ part, int n_w, int n_det, int max_exc,
                                                    int n_orb, int NP, int n_vtot) {
    extern __shared__ __align__(16) double2 Ss[];      // [CE_CH][NP*NP]
    __shared__ int tx_s[CE_CH], ty_s[CE_CH];
    const int chunk = blockIdx.x, w = blockIdx.y, tid = threadIdx.x;
    const long long t0 = (long long)chunk * CE_CH;
    const int nt = (int)min((long long)CE_CH, n_tiles - t0), NP2 = NP * NP;
    for (int i = tid; i < nt * NP2; i += 128) {
        const int tl = i / NP2;
        Ss[i] = S[((size_t)(t0 + tl) * n_w + w) * NP2 + (i - tl * NP2)];
    }
    if (tid < nt) { tx_s[tid] = tiles[t0 + tid].pi; ty_s[tid] = tiles[t0 + tid].pj; }
    __syncthreads();
    for (int d = tid; d < n_det; d += 128) {
        const size_t v = (size_t)w * n_det + d;
        const signed char* kd = kind + (size_t)d * n_orb;
        const int* hi = holeIdx + (size_t)d * max_exc;
        int e = 0;
        while (e < max_exc && hi[e] >= 0) ++e;
        const double2* Gv = G + v * max_exc * n_orb;
        double2 ek = make_double2(0.0, 0.0), ej = make_double2(0.0, 0.0);
        for (int tl = 0; tl < nt; ++tl) {
            const int x = tx_s[tl], y = ty_s[tl];
            const int kx = kd[x], ky = kd[y];
            if (kx < 0 || ky < 0) continue;
            const double2* St = Ss + tl * NP2;
            // coefficient lists: entry 0 = self (index 0 for the x role, 1 for the y role), entries 1..e = the holes
            double2 cx[MAXE + 1], cy[MAXE + 1];
            int ix[MAXE + 1], iy[MAXE + 1];
            cx[0] = make_double2(kx == 0 ? 1.0 : 0.0, 0.0); ix[0] = 0;
            cy[0] = make_double2(ky == 0 ? 1.0 : 0.0, 0.0); iy[0] = 1;
#pragma unroll
            for (int k = 0; k < MAXE; ++k) {
                const bool on = k < e;
                cx[1 + k] = on ? Gv[(size_t)k * n_orb + x] : make_double2(0.0, 0.0); ix[1 + k] = on ? 2 + hi[k] : 0;
                cy[1 + k] = on ? Gv[(size_t)k * n_orb + y] : make_double2(0.0, 0.0); iy[1 + k] = on ? 2 + hi[k] : 0;
            }
#pragma unroll
            for (int a = 0; a <= MAXE; ++a) {
                if (a > e) break;
#pragma unroll
                for (int b = 0; b <= MAXE; ++b) {
                    if (b > e) break;
                    const double2 cc = cmul(cy[a], cx[b]);
                    const double2 se = St[iy[a] * NP + ix[b]], sj = St[ix[b] * NP + iy[a]];
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
    const double2* Hw = H + (size_t)w * n_orb * 9;
    const double2* Gv = G + (size_t)v * max_exc * n_orb;
    for (int x = 0; x < n_orb; ++x) {
        if (kd[x] < 0) continue;
        if (kd[x] == 0) { e1.x += Hw[x * 9].x; e1.y += Hw[x * 9].y; }
        for (int k = 0; k < max_exc && hi[k] >= 0; ++k) {
            const double2 t1 = cmul(Gv[(size_t)k * n_orb + x], Hw[x * 9 + 1 + hi[k]]);
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

struct Timer {
    lo_factors* f;
    cudaStream_t s;
    int idx = -1;
    Timer(lo_factors* f_, cudaStream_t s_, int kind) : f(f_), s(s_) {
        if (!f->timing) return;
        TimingEvent ev;
        if (!f->pool.empty()) { ev = f->pool.back(); f->pool.pop_back(); }
        else { cudaEventCreate(&ev.e0); cudaEventCreate(&ev.e1); }
        ev.kind = kind;
        cudaEventRecord(ev.e0, s);
        f->events.push_back(ev);
        idx = (int)f->events.size() - 1;
    }
    ~Timer() { if (idx >= 0) cudaEventRecord(f->events[idx].e1, s); }
};

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
    e = cudaFuncSetAttribute(k_coulomb<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, CO_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_coulomb<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, CO_SMEM);
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
    e = cudaFuncSetAttribute(k_cas_pairs<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, CpCfg<4>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_pairs<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, CpCfg<6>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_cas_pairs<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, CpCfg<8>::SMEM);
    if (e != cudaSuccess) { set_error(std::string("cudaFuncSetAttribute(k_cas_*): ") + cudaGetErrorString(e)); return LO_ECUDA; }
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

lo_status launch_s3_s5(lo_factors* f, int n_w, void* E_L, void* E1, void* E_J, void* E_K, int* walker_status, void* Eout4, cudaStream_t stream);

lo_status launch_local_energy(lo_factors* f, int n_w, const void* phi_a, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K,
                              int* walker_status, void* Eout4, cudaStream_t stream) {
    const void* phis[2] = {phi_a, phi_b};
    for (int s = 0; s < f->n_spin; ++s)
        launch_s1(f, n_w, f->ops->dPsi[s], f->n_occ[s], f->n_occ[s], phis[s], f->dA[s], f->dStatus + (size_t)s * f->Wcap, f->dThT, f->o_base[s],
                  f->ldw, stream);
    return launch_s3_s5(f, n_w, E_L, E1, E_J, E_K, walker_status, Eout4, stream);
}

// S2-S5 on the Theta^T panels of n_w (possibly virtual, see lo_local_energy_cas) walkers.
lo_status launch_s3_s5(lo_factors* f, int n_w, void* E_L, void* E1, void* E_J, void* E_K, int* walker_status, void* Eout4, cudaStream_t stream) {
    const int N_pad = f->N_pad, ldw = f->ldw, Wcap = f->Wcap;
    const int NB = (n_w + WALKER_TILE - 1) / WALKER_TILE;
    // ---- S2 + S3
    const int RB = f->Xp / CO_BM;
    const int ksteps = f->O_tot * (N_pad / KTILE);
    const int nsplit = pick_split((long long)RB * NB, ksteps, f->num_sms);
    double2* EJpart = (double2*)f->dEJpart;
    double2* E1raw = EJpart + (size_t)RB * Wcap;
    {
        Timer tm(f, stream, LO_K_COULOMB);
        long long items = (long long)RB * NB * nsplit;
        int grid = (int)std::min<long long>(items, f->num_sms);
        if (n_w % WALKER_TILE)
            k_coulomb<true><<<grid, 384, CO_SMEM, stream>>>(f->ops->tmLbar, f->tmTheta, f->dXpart, f->Xp, f->O_tot, N_pad, ldw, RB, NB, nsplit, 2 * n_w);
        else
            k_coulomb<false><<<grid, 384, CO_SMEM, stream>>>(f->ops->tmLbar, f->tmTheta, f->dXpart, f->Xp, f->O_tot, N_pad, ldw, RB, NB, nsplit, 2 * n_w);
        dim3 g2(NB * 2, RB);
        k_ej<<<g2, 256, 0, stream>>>(f->dXpart, EJpart, E1raw, f->Xp, ldw, nsplit, f->n_chol, Wcap);
    }
    // ---- S4
    int ex_grid = 0;
    {
        Timer tm(f, stream, LO_K_EXCHANGE);
        const bool coul = f->coulomb_lo != 0;
        long long items = (coul ? f->n_tiles4 : f->n_tiles) * NB;
        ex_grid = (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
        const bool ragged = n_w % WALKER_TILE != 0;
        if (!coul && n_w <= 32) {
            // narrow batch: 16-walker column blocks, row fragments split over the warps
            const int NB16 = (n_w + 15) / 16;
            items = f->n_tiles * NB16;
            ex_grid = (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
            k_exchange_narrow<<<ex_grid, 384, EN_SMEM, stream>>>(f->tmU, f->tmW, f->tmU8, f->tmW8, f->tmTheta32, f->dWgt, f->dTiles, items, NB16,
                                                                 N_pad, ldw, f->dEKpart, Wcap);
        } else
#define LO_EX_LAUNCH(C_, R_, TILES_, EJ_)                                                                                              \
    k_exchange<C_, R_><<<ex_grid, 384, EX_SMEM, stream>>>(f->tmU, f->tmW, f->tmU8, f->tmW8, f->tmTheta, f->dWgt, TILES_, items, NB, N_pad, ldw, \
                                                          f->dEKpart, EJ_, Wcap, n_w)
        if (coul && ragged) LO_EX_LAUNCH(true, true, f->dTiles4, f->dEJLpart);
        else if (coul) LO_EX_LAUNCH(true, false, f->dTiles4, f->dEJLpart);
        else if (ragged) LO_EX_LAUNCH(false, true, f->dTiles, nullptr);
        else LO_EX_LAUNCH(false, false, f->dTiles, nullptr);
#undef LO_EX_LAUNCH
    }
    // ---- S5
    {
        Timer tm(f, stream, LO_K_FINAL);
        const double c1 = f->n_spin == 1 ? 2.0 : 1.0, cJ = f->n_spin == 1 ? 2.0 : 0.5;
        k_finalize<<<(n_w + 127) / 128, 128, 0, stream>>>(EJpart, RB, E1raw, (const double2*)f->dEKpart, ex_grid, f->dStatus, f->n_spin, Wcap,
                                                          n_w, c1, cJ, (double2*)E_L, (double2*)E1, (double2*)E_J, (double2*)E_K,
                                                          walker_status, (double2*)Eout4,
                                                          f->coulomb_lo ? (const double2*)f->dEJLpart : nullptr);
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
        if (n_w % WALKER_TILE)
            k_coulomb<true><<<grid, 384, CO_SMEM, stream>>>(ops.tmLt, f->tmXT, f->dB, (int)ops.tri_pad, 1, ops.Xk_pad, f->ldw, RB, NB, 1, 2 * n_w);
        else
            k_coulomb<false><<<grid, 384, CO_SMEM, stream>>>(ops.tmLt, f->tmXT, f->dB, (int)ops.tri_pad, 1, ops.Xk_pad, f->ldw, RB, NB, 1, 2 * n_w);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("lo_propagator: kernel launch failed: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

// local energy with a multi-determinant trial by direct summation over determinants (Eq. 12), the
// determinants' overlaps and Green's functions by SMW updates of the reference (Eq. 20); each (walker, determinant) is a
// virtual walker of the ordinary Coulomb / exchange kernels (orbital-indexed Theta^d panels, zero where unoccupied).
lo_status launch_local_energy_cas(lo_factors* f, int n_w, const void* phi, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K,
                                  void* ovlp, int* walker_status, cudaStream_t stream) {
    CasPlan& c = *f->cas;
    const int n_orb = f->n_occ[0], n_v = n_w * c.n_det, ldw0 = 2 * c.W0cap;
    launch_s1(f, n_w, f->ops->dPsi[0], n_orb, c.n_ref, phi, c.dA0, c.dSt0, c.dTh0, 0, ldw0, stream);
    k_cas_T<<<n_w, 256, 0, stream>>>(f->ops->dPsi[0], n_orb, c.dTh0, (double2*)c.dT, f->N, f->N_pad, c.n_ref, c.n_virt, ldw0);
    int* stv = c.mode == 0 ? f->dStatus : c.dStV;
    k_cas_coef<<<(n_v + 3) / 4, 128, 0, stream>>>((const double2*)c.dT, c.dHoles, c.dParts, c.dCoef, c.dSt0, (double2*)c.dG, (double2*)c.dWd,
                                                  stv, n_v, c.n_det, c.max_exc, c.n_ref, c.n_virt, n_orb, c.has_beta ? 1 : 0);
    if (c.has_beta) {
        // unrestricted trial: the beta strings get their own SMW data; their Theta^d panels follow the alpha panels
        const int n_orb_b = f->n_occ[1];
        launch_s1(f, n_w, f->ops->dPsi[1], n_orb_b, c.n_ref_b, phi_b, c.dA0B, c.dSt0B, c.dTh0B, 0, ldw0, stream);
        k_cas_T<<<n_w, 256, 0, stream>>>(f->ops->dPsi[1], n_orb_b, c.dTh0B, (double2*)c.dTB, f->N, f->N_pad, c.n_ref_b, c.n_virt_b, ldw0);
        k_cas_coef<<<(n_v + 3) / 4, 128, 0, stream>>>((const double2*)c.dTB, c.dHolesB, c.dPartsB, c.dCoef, c.dSt0B, (double2*)c.dGB,
                                                      (double2*)c.dWdB, f->dStatus + f->Wcap, n_v, c.n_det, c.max_exc, c.n_ref_b, c.n_virt_b,
                                                      n_orb_b, 2);
        dim3 g3b(n_v, n_orb_b, (f->N_pad + 127) / 128);
        k_cas_theta<<<g3b, 128, 0, stream>>>(c.dTh0B, (const double2*)c.dGB, c.dHolesB, f->dThT, f->N_pad, c.n_ref_b, n_orb_b, c.n_det, c.max_exc,
                                             ldw0, f->ldw, f->o_base[1]);
    }
    if (c.mode == 0) {
        dim3 g3(n_v, n_orb, (f->N_pad + 127) / 128);
        k_cas_theta<<<g3, 128, 0, stream>>>(c.dTh0, (const double2*)c.dG, c.dHoles, f->dThT, f->N_pad, c.n_ref, n_orb, c.n_det, c.max_exc, ldw0, f->ldw, 0);
        lo_status st = launch_s3_s5(f, n_v, nullptr, nullptr, nullptr, nullptr, nullptr, c.dEv, stream);
        if (st != LO_OK) return st;
    } else {
        // rearranged SMW energy (Eq. 23): S intermediates once per (tile, walker), then small per-determinant forms
        const int WB = (n_w + 7) / 8;
        const long long items = f->n_tiles * WB;
        const int grid = (int)std::min<long long>(std::max<long long>(items, 1), f->num_sms);
        const int* actd = c.dHoleIdx + (size_t)c.n_det * c.max_exc;      // A_set stored behind the hole indices
        if (c.NP == 4)
            k_cas_pairs<4><<<grid, 384, CpCfg<4>::SMEM, stream>>>(f->tmU, f->tmW, c.tmTh0, f->dWgt, f->dTiles, items, WB, f->N_pad, ldw0, actd, (double2*)c.dS, n_w);
        else if (c.NP == 6)
            k_cas_pairs<6><<<grid, 384, CpCfg<6>::SMEM, stream>>>(f->tmU, f->tmW, c.tmTh0, f->dWgt, f->dTiles, items, WB, f->N_pad, ldw0, actd, (double2*)c.dS, n_w);
        else
            k_cas_pairs<8><<<grid, 384, CpCfg<8>::SMEM, stream>>>(f->tmU, f->tmW, c.tmTh0, f->dWgt, f->dTiles, items, WB, f->N_pad, ldw0, actd, (double2*)c.dS, n_w);
        const double* hbar = f->ops->dLbar + (size_t)f->n_chol * f->O_tot * f->N_pad;
        k_cas_H<<<n_w, 256, 0, stream>>>(hbar, c.dTh0, actd, c.n_act, (double2*)c.dH, f->N, f->N_pad, c.n_ref, n_orb, ldw0);
        const int n_chunks = (int)((f->n_tiles + CE_CH - 1) / CE_CH);
        const int n_vtot = c.max_real * c.n_det;
        if (n_chunks > 0) {
            dim3 g4(n_chunks, n_w);
            const size_t sm4 = (size_t)CE_CH * c.NP * c.NP * 16;
            if (c.max_exc <= 2)
                k_cas_energy<2><<<g4, 128, sm4, stream>>>((const double2*)c.dS, f->dTiles, f->n_tiles, c.dKind, c.dHoleIdx, (const double2*)c.dG,
                                                          (double2*)c.dPart, n_w, c.n_det, c.max_exc, n_orb, c.NP, n_vtot);
            else if (c.max_exc <= 4)
                k_cas_energy<4><<<g4, 128, sm4, stream>>>((const double2*)c.dS, f->dTiles, f->n_tiles, c.dKind, c.dHoleIdx, (const double2*)c.dG,
                                                          (double2*)c.dPart, n_w, c.n_det, c.max_exc, n_orb, c.NP, n_vtot);
            else
                k_cas_energy<8><<<g4, 128, sm4, stream>>>((const double2*)c.dS, f->dTiles, f->n_tiles, c.dKind, c.dHoleIdx, (const double2*)c.dG,
                                                          (double2*)c.dPart, n_w, c.n_det, c.max_exc, n_orb, c.NP, n_vtot);
        }
        k_cas_e1sum<<<(n_v + 127) / 128, 128, 0, stream>>>((const double2*)c.dPart, n_chunks, (const double2*)c.dH, c.dKind, c.dHoleIdx,
                                                           (const double2*)c.dG, (double2*)c.dEv, n_v, c.n_det, c.max_exc, n_orb, n_vtot);
    }
    k_cas_combine<<<(n_w + 127) / 128, 128, 0, stream>>>((const double2*)c.dEv, (const double2*)c.dWd, stv, c.dSt0,
                                                         c.has_beta ? (const double2*)c.dWdB : nullptr, c.has_beta ? f->dStatus + f->Wcap : nullptr,
                                                         c.has_beta ? c.dSt0B : nullptr, n_w, c.n_det,
                                                         (double2*)E_L, (double2*)E1, (double2*)E_J, (double2*)E_K, (double2*)ovlp, walker_status);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error(std::string("lo_local_energy_cas: kernel launch failed: ") + cudaGetErrorString(e)); return LO_ECUDA; }
    return LO_OK;
}

}  // namespace lo
