// lo_internal.h -- internal definitions of liblo_afqmc.so (not part of the C ABI).
// Data layout in HBM:
//   thT   [O_tot][ldw][N_pad] f64   Theta^T: orbital panel o, column c = 2*w + {0:re,1:im}, basis index p fastest.
//                                   ldw = 2*Wcap, Wcap = max_walkers rounded up to 64; rows p>=N and walkers >= n_w are 0.
//   LbarD [Xp][O_tot][N_pad]  f64   rows g<n_chol: Lbar^g_ip; row n_chol: hbar; rest 0.  Xp = ceil128(n_chol+1).
//   U, W  [rows][N_pad]       f64   packed factor rows of all pairs, pairs sorted by rank (descending), every pair
//                                   padded to a multiple of 8 rows; 64 slack rows at the end.
//   wgt   [rows]              f64   -cK * m_ij * sigma_K  (0 on padding rows).
//   tiles [n_tiles]                 row tiles of the grouped GEMM: {row0, nfrag (valid 8-row fragments, 1..8), pi, pj}.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <memory>
#include <string>
#include <vector>

#include "../../include/lo_afqmc.h"

namespace lo {

constexpr int KTILE = 16;        // K tile (basis index p) of both GEMMs, in doubles
constexpr int WALKER_TILE = 64;  // walkers per column block (128 real columns)
constexpr int EX_BM = 64;        // rows (singular vectors) per exchange tile
constexpr int CO_BM = 128;       // rows (Cholesky vectors) per Coulomb tile
constexpr int MAX_SPLIT = 8;     // split-K partial buffers of the Coulomb GEMM
#define LO_HOST_CHUNKS 4         // walker chunks of lo_local_energy_host (copy/compute overlap)

// Tensor maps of one array for every box height 8, 16, .., 64 rows (passed to kernels as one __grid_constant__ parameter).
struct TmSet {
    CUtensorMap m[8];
};

struct ExTile {
    int row0;   // first packed row of the tile
    int nfrag;  // valid 8-row fragments in the tile (1..8)
    int pi;     // Theta panel (global orbital index) contracted with W  (orbital i)
    int pj;     // Theta panel contracted with U                         (orbital j)
};

void set_error(const std::string& s);
std::string& err_buf();

// Device-resident operands shared between a factor set and its re-truncations.
struct SharedOps {
    int device = -1;
    double* dLbar = nullptr;      // [Xp][O_tot][N_pad]
    CUtensorMap tmLbar;           // 2D [Xp][O_tot*N_pad], box 128 x 16, 128B swizzle
    double* dPsi[2] = {nullptr, nullptr};  // [N][O_s]
    // propagator operand (LO_SETUP_PROPAGATOR): Lt[r(p,q)][g] = L^g_pq for p<=q, [tri_pad][Xk_pad] f64, zero padded
    double* dLt = nullptr;
    CUtensorMap tmLt;             // 2D [tri_pad][Xk_pad], box 128 x 16, 128B swizzle
    long long tri = 0, tri_pad = 0;
    int Xk_pad = 0;
    std::vector<double> hLbar;    // host copy [n_chol][O_tot][N] (+ hbar as row n_chol), kept for host-only sets / retruncate on host
    ~SharedOps();
};

// Growable device array over one contiguous virtual address range (lo_mem.cu).
struct GrowBuf {
    void* base = nullptr;
    size_t reserved = 0, mapped = 0, chunk = 0;
    int device = -1;
    std::vector<unsigned long long> handles;   // CUmemGenericAllocationHandle of every mapped chunk
    lo_status reserve(int device, size_t max_bytes);
    lo_status ensure(size_t bytes);            // map (zero-filled) physical memory so that [0, bytes) is usable
    void release();
};

// One row-block copy of the packing step: r rows of N_pad doubles from src_row to dst_row.
struct GatherRec {
    long long src_row, dst_row;
    int r, pad_;
};

// One pair of the SMW-energy path: its <= 4-fragment tiles are tiles4[t0 .. t0 + nt); S is kept per pair, not per tile.
struct CasPair {
    int t0, nt, pi, pj;
};

// Multi-determinant trial (lo_set_cas_trial): determinants as excitation lists of the reference
// (= the first n_ref orbitals of the factor set's Psi), workspace for max_real real walkers; the n_det determinants of a
// real walker are laid out as n_det consecutive VIRTUAL walkers of the ordinary S3-S5 path.
constexpr int CAS_MAX_EXC = 8;
constexpr int CAS_MAX_ACT = 12;     // distinct hole columns per spin in LO_CAS_SMW_ENERGY (closed shell; 6 for unrestricted trials)
constexpr int CAS_HS = 1 + CAS_MAX_ACT;   // slots per orbital of the one-body intermediates H
struct CasPlan {
    int n_ref = 0, n_det = 0, max_exc = 0, n_virt = 0, max_real = 0, W0cap = 0;
    int *dHoles = nullptr, *dParts = nullptr;   // [n_det][max_exc]
    double* dCoef = nullptr;                    // [n_det]
    double* dTh0 = nullptr;                     // Theta0^T panels [n_ref][2*W0cap][N_pad]
    double* dA0 = nullptr;                      // [W0cap][n_ref][n_ref] complex
    double* dT = nullptr;                       // T = C_virt^T Theta0: [W0cap][n_virt][n_ref] complex
    double* dG = nullptr;                       // SMW coefficients [max_real*n_det][max_exc][n_orb] complex
    double* dWd = nullptr;                      // weights c_d det(T_d)^2: [max_real*n_det] complex
    double* dEv = nullptr;                      // per virtual walker {E_L,E1,E_J,E_K}: [max_real*n_det][4] complex
    int* dSt0 = nullptr;                        // [W0cap] status of the reference overlap
    int* dStV = nullptr;                        // [max_real*n_det] status per (walker, determinant), SMW-energy mode
    // ---- beta strings of an unrestricted trial (lo_set_cas_trial_beta; direct mode only); alpha uses the fields above
    bool has_beta = false;
    int n_ref_b = 0, n_virt_b = 0;
    int *dHolesB = nullptr, *dPartsB = nullptr;
    double *dTh0B = nullptr, *dA0B = nullptr, *dTB = nullptr, *dGB = nullptr, *dWdB = nullptr;
    int* dSt0B = nullptr;
    // ---- rearranged SMW energy (Eq. 23), mode 1
    int mode = 0;                               // 0: direct summation over virtual walkers, 1: SMW energy
    int n_act = 0, NP = 0;                      // active (hole) columns A_set, panel-set size NP = 2 + padded n_act (4, 6 or 8)
    int hAct[16] = {0};                         // A_set (orbital = reference column), padded with 0
    int* dHoleIdx = nullptr;                    // [n_det][max_exc]: index of hole k in A_set
    signed char* dKind = nullptr;               // [n_det][n_orb]: -1 unoccupied, 0 reference non-hole, 1+m particle m
    double* dS = nullptr;                       // S[tile][w][NP][NP] complex (Eq. 23 intermediates contracted over K)
    double* dH = nullptr;                       // one-body intermediates [W0cap][n_orb][CAS_HS] complex (self, A_set)
    double* dPart = nullptr;                    // [n_chunks][max_real*n_det][2] complex partial (E_K, E_J) sums
    int n_chunks = 0;
    CUtensorMap tmTh0;                          // Theta0^T panels [n_orb*2*W0cap][N_pad], box 32 x 16 (16 walkers)
    // ---- rearranged SMW energy with an UNRESTRICTED trial (n_spin == 2): the alpha data are the fields above, the beta
    // data the *B fields; exchange per spin from that spin's tiles, Coulomb by the Cholesky route from SMW-updated X^g
    int n_actB = 0, NPB = 0, n_chunksB = 0;
    int hActB[16] = {0};
    int* dHoleIdxB = nullptr;
    signed char* dKindB = nullptr;
    double *dSB = nullptr, *dHB = nullptr, *dPartB = nullptr;
    int* dStVB = nullptr;
    CUtensorMap tmTh0B;
    // more than 6 active columns (closed shell, <= CAS_MAX_ACT): the active set is cut into groups of gs = 3 and k_cas_pairs runs
    // once per pair of groups (a <= b) on the panel list {x, y, G_a, G_b}; pass p(a,b) = a ng - a(a-1)/2 + (b - a)
    int gs[2] = {6, 6}, ng[2] = {1, 1}, npass[2] = {1, 1}, ce[2] = {16, 16};   // group size, groups, passes, pairs per k_cas_energy chunk
    int* dPassAct[2] = {nullptr, nullptr};      // [npass][6] panel (orbital) indices of every pass
    CasPair* dPairs[2] = {nullptr, nullptr};    // pairs with rows, per spin (tile ranges into the factor set's <= 4-fragment tile list)
    long long npair[2] = {0, 0};
    double* dThAct[2] = {nullptr, nullptr};     // gathered active panels [n_act][2*W0cap][N_pad] per spin (A operand of the Z GEMM)
    double* dZ[2] = {nullptr, nullptr};         // Z[(a, 2w+c)][g*O_tot + o] = Lbar^g_o . Theta0_{A_a}: [n_act*2*W0cap][Xp*O_tot]
    CUtensorMap tmThAct[2];                     // [n_act*2*W0cap][N_pad], box 128 x 16
    CUtensorMap tmLbarRows;                     // Lbar as [(Xp*O_tot)][N_pad], box 128 x 16
    double* dEJu = nullptr;                     // [max_real*n_det] complex: E_J of every (walker, determinant)
};

// Pair-block SVD (lo_svd.cu)
constexpr int SVD_B = 16;            // rows per block (a subproblem = 2 blocks = 32 rows)
constexpr int SVD_MAX_SWEEPS = 40;
struct SvdStat {
    int sweeps = 0;          // sweeps performed (the last one only checks)
    double offdiag = 0;      // largest |g_p.g_q| / (|g_p||g_q|) over the non-null rows seen in the last sweep
    bool converged = true;
    long long screened = 0;  // blocks whose |Y|_F was <= the threshold: no iteration, rank 0
};

struct TimingEvent {
    cudaEvent_t e0, e1;
    int kind;
};

}  // namespace lo

struct lo_factors {
    int N = 0, N_pad = 0, n_chol = 0, Xp = 0, n_spin = 0, n_occ[2] = {0, 0}, O_tot = 0, o_base[2] = {0, 0};
    double threshold = 0;
    int device = -1, max_walkers = 0, Wcap = 0, ldw = 0, num_sms = 0;
    int setup_on_gpu = 0;
    lo::SvdStat svd_stat;                // worst case over all pair blocks of lo_setup
    double setup_seconds = 0, setup_svd_seconds = 0;
    long long n_rsvd_accepted = 0;       // pair blocks whose randomised sketch was accepted (LO_SETUP_RANDOMIZED_SVD)
    int rsvd_k = 0;                      // sketch size, 0 = full SVD only
    long long n_prescreened = 0;         // pairs the norm bound removed before their block was formed
    long long n_energy_screened = 0;     // pairs lo_screen_pairs dropped (m_ij sigma_1 <= energy_cutoff)
    double energy_cutoff = 0, energy_bound = 0;   // and cK * sum over them of m_ij sigma_1
    // pair bookkeeping, natural (row-major i<=j) order per spin
    std::vector<int> rank[2];
    std::vector<long long> row_off[2];   // first packed row of the pair
    std::vector<double> sigma_next[2];   // first discarded singular value of the pair (0 if none); for the truncation bound
    long long rows = 0;                  // packed rows incl. per-pair padding (without slack)
    long long n_tiles = 0;
    // host copies: hU/hW only for host-only sets (device < 0); hWgt (weights incl. sigma) always
    std::vector<double> hU, hW, hWgt;
    std::vector<lo::ExTile> hTiles;
    std::vector<lo::ExTile> hTiles4;     // same rows cut at <= 4 fragments (compressed-Coulomb mode, NEXT-3)
    long long n_tiles4 = 0;
    int coulomb_lo = 0;                  // 1: E_J from the compressed factors (Eq. 19/22) instead of the Cholesky route
    // device factor set
    lo::GrowBuf bU, bW;                  // backing store of dU / dW
    double *dU = nullptr, *dW = nullptr, *dWgt = nullptr;
    lo::ExTile* dTiles = nullptr;
    lo::ExTile* dTiles4 = nullptr;
    int *dSchedOff = nullptr, *dSchedTile = nullptr;   // static schedule of the tiles over num_sms CTAs (small problems), CSR
    CUtensorMap tmU, tmW, tmTheta;       // 2D [rows][N_pad]: boxes 64 x 16 (U, W) and 128 x 16 (Theta^T), 128B swizzle
    CUtensorMap tmU8, tmW8;              // same arrays, boxes 8 x 16 (one row fragment): tiles shorter than 64 rows
    lo::TmSet tmUf, tmWf;                // same arrays, boxes (8 k) x 16 for k = 1..8: one TMA issue per operand for a tile of k fragments
    CUtensorMap tmTheta32;               // Theta^T panels with a 32 x 16 box (16 walkers): narrow-batch exchange
    std::shared_ptr<lo::SharedOps> ops;
    // workspace
    double* dThT = nullptr;       // [O_tot][ldw][N_pad]
    double* dA[2] = {nullptr, nullptr};  // [Wcap][O_s][O_s] complex
    double* dXpart = nullptr;     // [MAX_SPLIT][Xp][ldw]
    double* dEJpart = nullptr;    // [Xp/128][Wcap] complex
    double* dEKpart = nullptr;    // [num_sms][Wcap] complex
    double* dEJLpart = nullptr;   // [num_sms][Wcap] complex (compressed-Coulomb partials)
    int* dStatus = nullptr;       // [2][Wcap]
    double* dEout = nullptr;      // [Wcap][4] complex (host variant)
    int* dStatusOut = nullptr;    // [Wcap]
    double* dPhi[2] = {nullptr, nullptr};  // staging for the host variant
    double* dXT = nullptr;        // propagator: fields as a K-major real operand [ldw][Xk_pad] (row 2w+c = re/im of walker w)
    double* dB = nullptr;         // propagator output [tri_pad][ldw] (= complex [tri_pad][Wcap])
    CUtensorMap tmXT;
    cudaStream_t copyStream = nullptr;     // host variant: H2D of walker chunk c+1 overlaps the kernels of chunk c
    cudaEvent_t evCopy[LO_HOST_CHUNKS] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t evEnter = nullptr;         // host variant: the copy stream waits for what the caller's stream already holds
    unsigned long long factor_bytes = 0, lbar_bytes = 0, workspace_bytes = 0;
    int last_n_w = 0;
    lo::CasPlan* cas = nullptr;
    // exchange on the tcgen05 tensor cores from INT8 digit slices (lo_set_exchange_mode, lo_exchange_i8.cu)
    int ex_mode = 0;                       // LO_EXCHANGE_DMMA / LO_EXCHANGE_INT8
    int8_t *dUq = nullptr, *dWq = nullptr; // [n_tiles][KB][7][64 x 32] digit slices of the factor rows
    int8_t* dThq = nullptr;                // [O_tot * Wcap/64][KB][7][128 x 32] digit slices of Theta^T, rewritten every call
    double* dWgtQ = nullptr;               // [rows + 64] wgt * 2^(eU + eW)
    double* dThScale = nullptr;            // [O_tot][Wcap] 2^e of the Theta rows
    double* dEKq = nullptr;                // [2 * num_sms][Wcap] complex partial sums
    double* dEJq = nullptr;                // same for the compressed Coulomb term (lo_set_coulomb_mode)
    int* dI8Fail = nullptr;
    int8_t* dLq = nullptr;                 // [Xp/64][O_tot][KB][7][64 x 32] digit slices of Lbar (rows g incl. hbar)
    int8_t* dLtq = nullptr;                // propagator: [tri_pad/64][KBx][7][64 x 32] digit slices of Lt (rows r(p,q), K = g)
    int* dELt = nullptr;                   // [tri_pad] exponents of the Lt rows
    int8_t* dXq = nullptr;                 // [Wcap/64][KBx][7][128 x 32] digit slices of the packed fields, rewritten every lo_propagator call
    double* dXScale = nullptr;             // [Wcap] 2^e of the field rows
    int* dELq = nullptr;                   // [O_tot][Xp] exponents of the (row g, orbital o) segments of Lbar
    unsigned long long i8_bytes = 0;
    // timing
    bool timing = false;
    std::vector<lo::TimingEvent> events;
    std::vector<lo::TimingEvent> pool;
    double t_ms[LO_K_COUNT] = {0};
    long long t_n[LO_K_COUNT] = {0};
};

namespace lo {

// hot path (lo_kernels.cu)
lo_status launch_local_energy(lo_factors* f, int n_w, const void* phi_a, const void* phi_b, void* E_L, void* E1, void* E_J,
                              void* E_K, int* walker_status, void* Eout4, cudaStream_t stream);
lo_status configure_kernels();
lo_status configure_cas_kernels();     // lo_cas.cu
// pieces of the hot path reused by the multi-determinant driver (lo_cas.cu)
void launch_s1(lo_factors* f, int n_w, const double* psi, int ldpsi, int O, const void* phi, double* dA, int* status, double* thT,
               int o_base, int ldw_t, cudaStream_t stream);
lo_status launch_s3_s5(lo_factors* f, int n_w, void* E_L, void* E1, void* E_J, void* E_K, int* walker_status, void* Eout4, cudaStream_t stream);
lo_status launch_propagator(lo_factors* f, int n_w, const void* x_dev, cudaStream_t stream);
// S3 alone on the Theta^T panels: X^g_w into f->dXpart (split-K partials summed into partial 0), E_J / E1 partials as a by-product.
void launch_coulomb_x(lo_factors* f, int n_w, cudaStream_t stream);
// out[r][c] = sum_p A[r][p] B[c][p] for K-major fp64 operands given as tensor maps with 128 x 16 boxes (rows, cols multiples
// of 128; ld_out >= cols): the Coulomb GEMM kernel on another pair of operands (Z intermediates of the unrestricted SMW energy).
void launch_gemm_kmajor(const CUtensorMap& tmA, const CUtensorMap& tmB, double* out, long long rows, long long cols, int N_pad, long long ld_out,
                        int num_sms, cudaStream_t stream);
lo_status launch_local_energy_cas(lo_factors* f, int n_w, const void* phi, const void* phi_b, void* E_L, void* E1, void* E_J, void* E_K, void* ovlp,
                                  int* walker_status, cudaStream_t stream);
// 2D fp64 tensor map over a row-major [rows][inner] array, box [box_rows][16], 128-byte swizzle, zero OOB fill.
lo_status make_tmap(CUtensorMap* tm, const void* base, unsigned long long inner, unsigned long long rows, unsigned box_rows);   // cudaFuncSetAttribute for the big-smem kernels (once per process/device)

// Pair-block SVD (lo_svd.cu): block one-sided Jacobi with Gram subproblems, host and device versions.
std::vector<int> svd_schedule(int n_blocks);
void host_block_svd(int R, int len, double* G, double* V, std::vector<double>& sigma, std::vector<int>& order, double skip_below, SvdStat* stat);
cudaError_t launch_block_jacobi(double* G, double* V, int n_mat, int n, int len, int ld, int ldv, const int* dSched, double skip_below, int* dSweeps,
                                double* dOff, const int* dIdx, size_t stride, cudaStream_t stream);

// Counter-based standard normal numbers for the test matrix of the randomised SVD: SplitMix64 of (seed + index) gives two
// uniforms, Box-Muller one Gaussian.  Host and device versions are the same function.
#ifdef __CUDACC__
__host__ __device__
#endif
inline double gauss_at(unsigned long long seed, unsigned long long index) {
    unsigned long long z = seed + 0x9E3779B97F4A7C15ull * (2 * index + 1);
    unsigned long long u[2];
    for (int r = 0; r < 2; ++r) {
        z += 0x9E3779B97F4A7C15ull;
        unsigned long long y = z;
        y = (y ^ (y >> 30)) * 0xBF58476D1CE4E5B9ull;
        y = (y ^ (y >> 27)) * 0x94D049BB133111EBull;
        u[r] = y ^ (y >> 31);
    }
    const double a = ((double)(u[0] >> 11) + 0.5) * (1.0 / 9007199254740992.0);      // (0, 1)
    const double b = ((double)(u[1] >> 11)) * (1.0 / 9007199254740992.0);            // [0, 1)
    return sqrt(-2.0 * log(a)) * cos(6.283185307179586 * b);
}

// GPU setup (lo_setup_gpu.cu): pair Gram matrices + block-Jacobi SVD (lo_svd.cu) for a batch of pairs of one spin.
// For the n listed pairs: returns sigma (descending, [n][N]) on the host and leaves the sorted U/W rows on the
// device in tmpU/tmpW ([n][N][N_pad]).  tmpY/tmpV are scratch of the same size.
lo_status gpu_pair_svd(const lo_factors* f, int spin, const int* pi, const int* pj, int n, double* tmpY, double* tmpV,
                       double* tmpU, double* tmpW, double* dSigma, int* dOrder, double* hSigma, double skip_below, SvdStat* stat);
size_t gpu_pair_svd_bytes_per_pair(int N, int N_pad);
// Randomised variant (LO_SETUP_RANDOMIZED_SVD): sketch of k rows, a-posteriori residual check, full method for the blocks
// the sketch does not capture; *n_accepted counts the blocks whose sketch was accepted.
lo_status gpu_pair_rsvd(const lo_factors* f, int spin, const int* pi, const int* pj, int n, int k, double* tmpY, double* tmpV, double* tmpU,
                        double* tmpW, double* dSigma, int* dOrder, double* hSigma, double skip_below, SvdStat* stat, long long* n_accepted);
// Host version for one pair block G (N x N, rows = columns of Y): returns true and the factors (sigma [k], U rows, W rows,
// k x N each) when the sketch is accepted.
bool host_pair_rsvd(int N, int k, const double* G, std::vector<double>& sigma, std::vector<double>& U, std::vector<double>& W, SvdStat* stat);
// dst[rec.dst_row + K][:] = src[rec.src_row + K][:] for K < rec.r, every rec of the host table (rows of N_pad doubles).
lo_status gpu_gather_rows(const double* src, double* dst, const GatherRec* table, int n, int N_pad);

// exchange from INT8 digit slices on tcgen05 (lo_exchange_i8.cu)
lo_status build_exchange_i8(lo_factors* f);
void free_exchange_i8(lo_factors* f);
void launch_slice_theta_i8(lo_factors* f, int n_w, cudaStream_t stream);
int launch_coulomb_i8(lo_factors* f, int n_w, cudaStream_t stream);
void launch_propagator_i8(lo_factors* f, int n_w, cudaStream_t stream);
void launch_exchange_i8(lo_factors* f, int n_w, cudaStream_t stream, bool coul, const double** part, int* n_part, const double** partJ);

// microbenchmarks (lo_peak.cu)
lo_status measure_peak(int device, int kind, double* value);
// gated experiment (lo_int8_probe.cu): FP64-accurate tile from INT8 slices on tcgen05; time per 128 x 128 x 384 tile, error vs fp64
lo_status measure_int8_slicing(int device, double* us_per_tile, double* max_err);

}  // namespace lo
